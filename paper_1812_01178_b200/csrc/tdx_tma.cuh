// tdx_tma.cuh -- x sweeps (unit-stride lines) through the Tensor Memory Accelerator.
//
// A unit-stride line of n = P*M doubles is a [P, M] matrix of partitions whose rows are M*8 = 128 bytes (M = 16) or
// 64 bytes (M = 8); the whole field is therefore a [lines*P, M] matrix with a contiguous row pitch.  One
// cp.async.bulk.tensor load brings a box of up to 256 such rows (32 KB, one contiguous piece of HBM) into shared memory
// with the 128B (64B) swizzle, so thread = partition reads ITS OWN row with eight (four) conflict-free 16-byte
// shared-memory loads: the "transpose" the unit-stride direction needs (PAPER.md:L51-74 is what the method removes) is
// done by the TMA address generator, not by load/store instructions.  The thread then runs Eq.(5) forward/backward in
// registers, trades interface values through shared memory, solves its rows of the reduced system (Eq.(7)), applies
// Eq.(8) (+ the Sherman-Morrison closure for periodic lines), writes the row back into the same swizzled slot, and one
// thread issues the TMA store.  A second bulk-tensor instruction per CTA prefetches into L2 the box that a CTA `pf`
// launches later will load, so HBM latency is paid one wave ahead and a few resident CTAs per SM keep HBM busy.
//
// HBM traffic: 8 B read + 8 B written per grid value; tables come from L1/L2.
// PAPER.md references: Eq.(5)-(8) L104-124, PDD L148-154, PPT L126-146/L156, Algorithm 1 steps 3,5,7 L240-258.
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>
#include "tdx_plan.cuh"
#include "tdx_kernels.cuh"

namespace tdx {

// ---- PTX helpers: mbarrier, TMA (cp.async.bulk.tensor), proxy fence ------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tm, const void* src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_prefetch_2d(const CUtensorMap* tm, int c0, int c1) {
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global [%0, {%1, %2}];"
                 ::"l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void tma_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tm)) : "memory");
}

// ---- unit-stride direction ------------------------------------------------------------------------------------
struct UnitTmaArgs {
    long long total_rows;    // tile rows in the field: lines * P * (tile rows per partition)
    int rows_per_cta;        // partitions per CTA = LPB * P (whole lines)
    int box_rows;            // tile rows per TMA box (<= 256); a CTA moves nbox boxes
    int nbox;
    int pf;                  // L2 prefetch distance in CTAs (0 = off)
};

constexpr int unit_tma_regs(int M) { return M <= 8 ? 56 : (M <= 16 ? 80 : 128); }

// The uniform row table (all partitions identical: uniform grid in x) travels as a kernel parameter (UniTable,
// tdx_kernels.cuh).

// M = rows per partition = doubles per partition row (16 -> 128-byte rows / SWIZZLE_128B, 8 -> 64-byte / SWIZZLE_64B,
// 32 -> two 128-byte tile rows per partition: eight lanes then hit four distinct swizzle keys, a 2-way bank conflict that
// the otherwise idle shared-memory pipe absorbs).
// UNI: one table for every partition (rows[jj*6+f], warp-uniform); else per-partition columns (rows[(jj*6+f)*P + p]).
template <int M, bool UNI, bool CYC>
__global__ void __maxnreg__(unit_tma_regs(M))
k_unit_tma(const __grid_constant__ CUtensorMap tmap, UnitTmaArgs A, Tables T, const __grid_constant__ UniTable<M> U) {
    extern __shared__ __align__(1024) unsigned char tma_smem[];
    constexpr int CH = M / 2;                                         // 16-byte chunks per partition
    constexpr int RPP = (M > 16) ? M / 16 : 1;                        // 128-byte tile rows per partition
    constexpr int CHR = CH / RPP;                                     // chunks per tile row (8, or 4 for M = 8)
    double2* tile = reinterpret_cast<double2*>(tma_smem);             // [blockDim.x * RPP][CHR] 16-byte chunks, hardware-swizzled
    const int rows_alloc = blockDim.x;                                 // partitions; >= rows_per_cta (multiple of 32)
    double* rf = reinterpret_cast<double*>(tile + (size_t)rows_alloc * CH);   // xt_first per partition
    double* rl = rf + rows_alloc;                                              // xt_last per partition
    uint64_t* bar = reinterpret_cast<uint64_t*>(rl + rows_alloc);
    const int r = threadIdx.x;
    const long long row0 = (long long)blockIdx.x * A.rows_per_cta * RPP;       // first tile row of this CTA

    if (r == 0) {
        if (smem_u32(tma_smem) & 1023u) __trap();                     // the hardware swizzle pattern assumes a 1024-byte aligned tile
        prefetch_tmap(&tmap);
        mbar_init(bar, 1);
        mbar_fence_init();
        mbar_arrive_expect_tx(bar, (uint32_t)(A.nbox * A.box_rows) * CHR * 16u);
        for (int b = 0; b < A.nbox; ++b) tma_load_2d(tile + (size_t)b * A.box_rows * CHR, &tmap, 0, (int)(row0 + (long long)b * A.box_rows), bar);
        if (A.pf > 0) {
            const long long prow = row0 + (long long)A.pf * A.rows_per_cta * RPP;
            if (prow < A.total_rows)
                for (int b = 0; b < A.nbox; ++b) tma_prefetch_2d(&tmap, 0, (int)(prow + (long long)b * A.box_rows));
        }
    }
    __syncthreads();                                                  // barrier initialised before anyone waits on it
    const int P = T.P;
    const int ll = r / P, p = r - ll * P;
    const bool valid = r < A.rows_per_cta;
    const double* rows = T.rows;
    auto tab = [&](int jj, int f) -> double {
        if (UNI) return U.v[jj * 6 + f];
        return __ldg(rows + ((size_t)jj * 6 + f) * P + (valid ? p : 0));
    };
    mbar_wait(bar, 0);

    double x[M];
    double2* myrow = tile + (size_t)r * CH;
    // SWIZZLE_128B: chunk ^= tile row & 7 (128-byte rows); SWIZZLE_64B: chunk ^= (tile row >> 1) & 3 (64-byte rows)
    auto slot = [&](int c) -> int {
        const int trow = r * RPP + c / CHR;
        const int key = (M == 8) ? ((trow >> 1) & 3) : (trow & 7);
        return (c / CHR) * CHR + ((c % CHR) ^ key);
    };
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        const double2 t = myrow[slot(c)];
        x[2 * c] = t.x; x[2 * c + 1] = t.y;
    }
    // Eq.(5): forward y_j = d_j - l_j y_{j-1}, backward xt_j = y_j inv_j - cp_j xt_{j+1}
#pragma unroll
    for (int jj = 1; jj < M; ++jj) x[jj] = fma(-tab(jj, F_L), x[jj - 1], x[jj]);
    x[M - 1] *= tab(M - 1, F_INV);
#pragma unroll
    for (int jj = M - 2; jj >= 0; --jj) x[jj] = fma(-tab(jj, F_CP), x[jj + 1], x[jj] * tab(jj, F_INV));
    rf[r] = x[0]; rl[r] = x[M - 1];
    __syncthreads();
    // Eq.(7): the two interface unknowns this partition needs
    double yL = 0.0, yR = 0.0, sc = 0.0;
    if (valid) {
        const int2 bd = __ldg(&T.band[p]);
        const double2* g2 = reinterpret_cast<const double2*>(T.G) + p;
        const int lb = ll * P;
        for (int k = 0; k < bd.y; ++k) {
            int idx = bd.x + k;
            if (idx >= 2 * P) idx -= 2 * P;                              // band may wrap (periodic line closed inside Z)
            const double rv = (idx & 1) ? rl[lb + (idx >> 1)] : rf[lb + (idx >> 1)];
            const double2 ab = __ldg(g2 + (size_t)k * P);                // {gL, gR}
            yL = fma(ab.x, rv, yL);
            yR = fma(ab.y, rv, yR);
        }
        if (CYC) {
            const int ns = __ldg(&T.Sn[0]);
            for (int k = 0; k < ns; ++k) {
                const int idx = __ldg(&T.Sidx[k]);
                const double rv = (idx & 1) ? rl[lb + (idx >> 1)] : rf[lb + (idx >> 1)];
                sc = fma(__ldg(&T.Sval[k]), rv, sc);
            }
        }
    }
    // Eq.(8): x = xt - v yL - w yR (- q s for periodic lines), back into the same swizzled slot
#pragma unroll
    for (int jj = 0; jj < M; ++jj) {
        double v = fma(-tab(jj, F_V), yL, x[jj]);
        v = fma(-tab(jj, F_W), yR, v);
        if (CYC) v = fma(-tab(jj, F_Q), sc, v);
        x[jj] = v;
    }
#pragma unroll
    for (int c = 0; c < CH; ++c) myrow[slot(c)] = make_double2(x[2 * c], x[2 * c + 1]);
    fence_proxy_async();                                              // generic-proxy writes -> visible to the TMA store
    __syncthreads();
    if (r == 0) {
        for (int b = 0; b < A.nbox; ++b) tma_store_2d(&tmap, tile + (size_t)b * A.box_rows * CHR, 0, (int)(row0 + (long long)b * A.box_rows));
        tma_commit();
        tma_wait_read<0>();                                           // shared memory must outlive the store's reads
    }
}

}  // namespace tdx
