// tdx_kernels.cuh -- the hot path: one launch per sweep, 8 B read + 8 B written per grid value.
//
//   k_strided<MAXM,V,CYC,UNI,REGS>  (UNI: one row table for every partition, passed as a kernel parameter; REGS: register budget)
//                          y / z sweeps and the Helmholtz y-solves: thread = (line, partition), a warp holds
//                          consecutive lines of ONE partition, so every global access is a coalesced row segment and
//                          the plan tables are warp-uniform.  Each thread keeps its partition (<= MAXM rows, V lines)
//                          in registers: forward + backward elimination (Eq.(5)), interface values to shared memory,
//                          reduced system (Eq.(7); PDD 2x2 blocks or PPT banded Z^{-1} rows), correction (Eq.(8)),
//                          Sherman-Morrison closure for periodic lines -- then one coalesced store.
//   k_unit<MAXM,UNI,CYC>   x sweeps (unit-stride lines): thread = partition, consecutive partitions in consecutive
//                          lanes; a warp's 32 partitions are one contiguous chunk of memory which is loaded coalesced,
//                          transposed through a padded per-warp shared-memory tile, and stored back the same way --
//                          no global transpose (PAPER.md:L51-74 is what the method removes).
//   k_thomas_strided / k_thomas_unit_tiled   mode THOMAS: one thread per line, plain recurrence, in place (GPU baseline).
//
// PAPER.md references: Eq.(5)-(8) L104-124, PDD L148-154, PPT L126-146/L156, Algorithm 1 steps 3,5,7 L240-258.
#pragma once
#include <cuda_runtime.h>
#include "tdx_plan.cuh"

namespace tdx {

struct Tables {
    const double* rows;      // row table (layout depends on the kernel), fields {l, q, inv, cp, v, w}
    const double* G;         // reduced coefficients, pairs {gL, gR}: G[g_index(set, side, k, p, KB, P)]
    const int2* band;        // band[set*P + p] = {lo, cnt} in interface-rhs indices r[0..2P)
    const int* Sidx;         // cyclic closure functional (sparse), Sidx/Sval[set*Scap + k], Sn[set]
    const double* Sval;
    const int* Sn;
    const double* pcr;       // PPT by plan-time cyclic reduction (k_pcr_tables): pcr[((set*pcr_cap + step)*P + p)*6 + f]; NULL = band of Z^-1 rows
    const int* pcr_n;        // exchange steps per set
    int pcr_cap;
    int P, n, q, r, KB, Scap;   // P: kernel partitions; q, r: the CALLER's partition map (n / Pu, n % Pu)
    int S;                      // sub-partitions per caller's partition (sub_part; 1 = plain map)
};

struct StridedArgs {
    double* data;            // base of the field (doubles)
    long long W;             // lines per outer index, in V-vectors
    long long line_stride;   // distance between consecutive rows of a line, in V-vectors
    long long outer_stride;  // distance between outer indices, in V-vectors
    int set_per_outer;       // 1: table set = set0 + outer index (Helmholtz wavenumber), 0: one set
    int set0;                // first set of this launch (a launch may cover a sub-range of the wavenumbers)
    int LPC;                 // lines (V-vectors) per CTA = blockDim.x
    int pf;                  // L2 prefetch distance: CTAs ahead (one tile per CTA) or sets ahead (looping CTAs); 0 = off
    int tiles_x;             // column tiles per outer index
    int tables_smem;         // 1: the TS instantiation (set's tables staged in shared memory)
    int pcr;                 // 1: the PCR instantiation (Tables::pcr)
    double* iface;           // slab sweeps (tdx_slab_eliminate): also store row 0 of every line to iface[0][outer][W*V] and its last
    long long iface_plane;   //   row to iface[1][...] (Alg.1 step 4's pack, fused into the store); iface_plane = doubles per plane; NULL = off
};

template <int V> struct VecIO;
template <> struct VecIO<1> {
    __device__ static inline void ld(const double* p, double (&x)[1]) { x[0] = __ldcs(p); }
    __device__ static inline void st(double* p, const double (&x)[1]) { __stcs(p, x[0]); }
};
template <> struct VecIO<2> {
    __device__ static inline void ld(const double* p, double (&x)[2]) { double2 t = __ldcs(reinterpret_cast<const double2*>(p)); x[0] = t.x; x[1] = t.y; }
    __device__ static inline void st(double* p, const double (&x)[2]) { __stcs(reinterpret_cast<double2*>(p), make_double2(x[0], x[1])); }
};

// Register budget per thread: the partition (MAXM x V doubles = 2 MAXM V registers) plus ~50 for addresses, table
// values in flight and the interface unknowns.  Measured on B200 (development sweeps): spills cost more than
// occupancy, and 2-4 small co-resident CTAs per SM beat one large one.
constexpr int strided_regs(int MAXM, int V) {
    return (MAXM * V <= 8) ? 64 : ((MAXM * V <= 16) ? 104 : ((MAXM * V <= 32) ? 128 : ((MAXM * V <= 48) ? 168 : 255)));
}
constexpr int strided_block_threads(int MAXM, int V) {            // largest CTA the register budget allows
    return (65536 / strided_regs(MAXM, V)) / 32 * 32 > 1024 ? 1024 : (65536 / strided_regs(MAXM, V)) / 32 * 32;
}

// A row table shared by every partition (uniform grid: all blocks A_p identical) travels as a kernel parameter: with the
// row loops fully unrolled every table value is a constant-bank operand of its DFMA -- no load instruction, no L1
// wavefront, no register holding a table value in flight.
template <int M> struct UniTable { double v[M * 6]; };

// UNI: row table = U.v[jj*6 + f] for every partition (ROWS_U plans: periodic or interior-identical blocks, one set).
// REGS: register budget; the default is the tier of the partition size, a smaller one buys a wider CTA (longer row segments).
// TS (one table set per outer index = the Helmholtz y-solves): the CTA copies its set's row table and reduced-system
// coefficients into shared memory once, before its tiles; every table read of the three passes and of the band loop is
// then an LDS (two addresses per warp, partitions padded by 16 bytes: conflict-free) instead of an L1 hit competing with
// the tile's own loads and stores in the L1TEX pipe.
// PCR (PPT, non-periodic lines): the reduced system is solved by block cyclic reduction with plan-time coefficients
// (k_pcr_tables, tdx_plan.cuh) instead of the 2P-term band of Z^-1 rows: ceil(log2(P-1)) steps of six multiply-adds per line,
// one barrier each, right-hand sides exchanged through double-buffered shared memory.
template <int MAXM, int V, bool CYC, bool UNI, int REGS = strided_regs(MAXM, V), bool TS = false, bool PCR = false>
__global__ void __maxnreg__(REGS)
k_strided(StridedArgs A, Tables T, const __grid_constant__ UniTable<UNI ? MAXM : 1> U) {
    static_assert(!(PCR && (TS || CYC || UNI)), "PCR is built for the plain per-set tables only");
    extern __shared__ double rs[];                          // rs[(idx*LPC + tx)*V + v], idx in [0, 2P)
    const int tx = threadIdx.x, p = threadIdx.y;
    const int LPC = A.LPC, P = T.P;
    const int o = blockIdx.y;
    const int set = A.set_per_outer ? A.set0 + o : 0;
    constexpr int RSTR = MAXM * 3 + 1;                      // TS: double2 per partition in shared memory (padded)
    double2* const st_rows = reinterpret_cast<double2*>(rs + (size_t)2 * P * LPC * V);
    double2* const st_G = st_rows + (size_t)P * RSTR;
    if (TS) {
        const int tid = p * LPC + tx, nth = LPC * P;
        const double2* src = reinterpret_cast<const double2*>(T.rows + (size_t)set * P * MAXM * 6);
        for (int k = tid; k < P * MAXM * 3; k += nth) { const int pp = k / (MAXM * 3); st_rows[pp * RSTR + (k - pp * MAXM * 3)] = __ldg(src + k); }
        const double2* gsrc = reinterpret_cast<const double2*>(T.G) + (size_t)set * T.KB * P;
        for (int k = tid; k < T.KB * P; k += nth) st_G[k] = __ldg(gsrc + k);
        __syncthreads();
    }
    const double2* const trow = st_rows + p * RSTR;
    int start, m;
    sub_part(p, T.q, T.r, T.S, start, m);
    const bool full = (T.r == 0) && (T.q == MAXM * T.S);    // every partition has exactly MAXM rows (warp-uniform)
    const long long rstride = A.line_stride * V;
    // One table set per outer index (Helmholtz: a set per wavenumber): this CTA's set is cold in L1, so pull its lines
    // in now, one prefetch per thread -- otherwise every table load on the dependent chain and in the band loop pays
    // L2 latency.  Such a CTA then works through several column tiles of its set (the loop below) with warm tables.
    if (A.set_per_outer && !TS) {
        const int tid = p * LPC + tx, nth = LPC * P;
        const char* rb = reinterpret_cast<const char*>(T.rows + (size_t)set * P * MAXM * 6);
        const int rlines = (P * MAXM * 48 + 127) >> 7;
        for (int k = tid; k < rlines; k += nth) asm volatile("prefetch.global.L1 [%0];" ::"l"(rb + ((size_t)k << 7)));
        const char* gb = reinterpret_cast<const char*>(T.G + (size_t)set * 2 * T.KB * P);
        const int glines = (2 * T.KB * P * 8 + 127) >> 7;
        for (int k = tid; k < glines; k += nth) asm volatile("prefetch.global.L1 [%0];" ::"l"(gb + ((size_t)k << 7)));
    }
    const double2* rt = reinterpret_cast<const double2*>(T.rows + ((size_t)((size_t)set * P + p) * MAXM) * 6);
    const int tiles_x = A.tiles_x;

  // column tiles of this CTA: exactly one when gridDim.x == tiles_x, else blockIdx.x, blockIdx.x + gridDim.x, ...
  for (int xt = blockIdx.x; xt < tiles_x; xt += gridDim.x) {
    const long long i = (long long)xt * LPC + tx;
    const bool valid = i < A.W;
    double* base = A.data + ((long long)o * A.outer_stride + (long long)start * A.line_stride + i) * V;

    double x[MAXM][V];
#pragma unroll
    for (int jj = 0; jj < MAXM; ++jj) {
        if (valid && (full || jj < m)) VecIO<V>::ld(base + jj * rstride, x[jj]);
        else {
#pragma unroll
            for (int v = 0; v < V; ++v) x[jj][v] = 0.0;
        }
    }
    // L2 prefetch of a tile that is loaded later -- by the CTA `pf` launches ahead (one tile per CTA), or by this CTA
    // in its next iteration / by the CTA `pf` sets ahead (looping CTAs): one lane per 128-byte line.  Whoever needs the
    // data then finds it in L2 (~300 cycles) instead of HBM, so a few resident CTAs per SM keep HBM busy.
    if (A.pf > 0 && ((tx * V) & 15) == 0) {
        int nbx, nby;
        if ((int)gridDim.x == tiles_x) {
            const long long lin = (long long)o * tiles_x + xt + A.pf;
            nby = (int)(lin / tiles_x); nbx = (int)(lin - (long long)nby * tiles_x);
        } else {
            nbx = xt + gridDim.x; nby = o;
            if (nbx >= tiles_x) { nbx = blockIdx.x; nby = o + A.pf; }
        }
        const long long ip = (long long)nbx * LPC + tx;
        if (nby < (int)gridDim.y && ip < A.W) {
            const double* pb = A.data + ((long long)nby * A.outer_stride + (long long)start * A.line_stride + ip) * V;
#pragma unroll
            for (int jj = 0; jj < MAXM; ++jj)
                if (full || jj < m) asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + jj * rstride));
        }
    }

    // Eq.(5): forward y_j = d_j - l_j y_{j-1}, backward xt_j = y_j inv_j - cp_j xt_{j+1}
#pragma unroll
    for (int jj = 1; jj < MAXM; ++jj) {
        const double l = UNI ? U.v[UNI ? jj * 6 + F_L : 0] : (TS ? trow[jj * 3 + 0].x : __ldg(reinterpret_cast<const double*>(&rt[jj * 3 + 0])));
#pragma unroll
        for (int v = 0; v < V; ++v) x[jj][v] = fma(-l, x[jj - 1][v], x[jj][v]);
    }
    {
        const double inv = UNI ? U.v[UNI ? (MAXM - 1) * 6 + F_INV : 0] : (TS ? trow[(MAXM - 1) * 3 + 1].x : __ldg(reinterpret_cast<const double*>(&rt[(MAXM - 1) * 3 + 1])));
#pragma unroll
        for (int v = 0; v < V; ++v) x[MAXM - 1][v] *= inv;
    }
#pragma unroll
    for (int jj = MAXM - 2; jj >= 0; --jj) {
        const double2 ic = UNI ? make_double2(U.v[UNI ? jj * 6 + F_INV : 0], U.v[UNI ? jj * 6 + F_CP : 0]) : (TS ? trow[jj * 3 + 1] : __ldg(&rt[jj * 3 + 1]));   // {inv, cp}
#pragma unroll
        for (int v = 0; v < V; ++v) x[jj][v] = fma(-ic.y, x[jj + 1][v], x[jj][v] * ic.x);
    }
    // E^T xt: first and last row of this partition
#pragma unroll
    for (int v = 0; v < V; ++v) {
        rs[((2 * p) * LPC + tx) * V + v] = x[0][v];
        rs[((2 * p + 1) * LPC + tx) * V + v] = x[MAXM - 1][v];  // xt_last (padding rows carry it to the last slot)
    }
    __syncthreads();
    // Eq.(7): the two interface unknowns this partition needs
    double yL[V], yR[V], sc[V];
#pragma unroll
    for (int v = 0; v < V; ++v) { yL[v] = 0.0; yR[v] = 0.0; sc[v] = 0.0; }
    if (PCR) {
        // block p = (s_p, t_p) = (x_last of partition p-1, x_first of partition p), p = 1..P-1; thread 0 only takes part in the barriers
        double* pb = rs + (size_t)2 * P * LPC * V;          // 2 buffers x {q0, q1} x [P][LPC*V]
        const int S2 = P * LPC * V, me = (p * LPC + tx) * V;
        const int nst = __ldg(&T.pcr_n[set]);
        const double2* pc = reinterpret_cast<const double2*>(T.pcr) + ((size_t)set * T.pcr_cap * P + p) * 3;
        double r0[V], r1[V], q0[V], q1[V];
#pragma unroll
        for (int v = 0; v < V; ++v) {
            r0[v] = (p >= 1) ? rs[((2 * p - 1) * LPC + tx) * V + v] : 0.0;   // xt_last of partition p-1
            r1[v] = (p >= 1) ? x[0][v] : 0.0;                                  // xt_first of this partition
        }
        for (int s = 0, d = 1;; ++s, d <<= 1) {
            const double2 c0 = __ldg(pc + (size_t)s * P * 3), c1 = __ldg(pc + (size_t)s * P * 3 + 1), c2 = __ldg(pc + (size_t)s * P * 3 + 2);
#pragma unroll
            for (int v = 0; v < V; ++v) {                   // D^-1 r: {idet, -beta idet}, {-gamma idet, l}, {u, -}
                q0[v] = fma(c0.y, r1[v], c0.x * r0[v]);
                q1[v] = fma(c1.x, r0[v], c0.x * r1[v]);
            }
            double* B = pb + (size_t)(s & 1) * 2 * S2;
            if (s == nst) {                                 // decoupled: s_p = q0 (own), t_{p+1} = q1 of the next block
#pragma unroll
                for (int v = 0; v < V; ++v) B[S2 + me + v] = q1[v];
                __syncthreads();
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    yL[v] = q0[v];
                    yR[v] = (p <= P - 2) ? B[S2 + me + LPC * V + v] : 0.0;
                }
                break;
            }
#pragma unroll
            for (int v = 0; v < V; ++v) { B[me + v] = q0[v]; B[S2 + me + v] = q1[v]; }
            __syncthreads();
            const int mL = ((p - d > 0 ? p - d : 0) * LPC + tx) * V, mR = ((p + d < P - 1 ? p + d : P - 1) * LPC + tx) * V;   // l, u are 0 beyond the ends
#pragma unroll
            for (int v = 0; v < V; ++v) {
                r0[v] = fma(-c1.y, B[mL + v], r0[v]);
                r1[v] = fma(-c2.x, B[S2 + mR + v], r1[v]);
            }
        }
    } else {
        const int2 bd = __ldg(&T.band[set * P + p]);
        const double2* g2 = reinterpret_cast<const double2*>(T.G) + (size_t)set * T.KB * P + p;
        auto term = [&](int k) {
            const double2 ab = TS ? st_G[k * P + p] : __ldg(g2 + (size_t)k * P);   // {gL, gR}
            const double a = ab.x, b = ab.y;
            int idx = bd.x + k;                             // band may wrap around (periodic line closed inside Z)
            if (idx >= 2 * P) idx -= 2 * P;
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const double rv = rs[(idx * LPC + tx) * V + v];
                yL[v] = fma(a, rv, yL[v]);
                yR[v] = fma(b, rv, yR[v]);
            }
        };
        // two band terms per iteration let the loads of the next term overlap the FMAs (cfg5 y 1.48 -> 1.44 ms); the
        // 255-register tile keeps the compiler's own choice, 4 (forcing 2 there: cfg4 Helmholtz 0.388 -> 0.399 ms, 1: 0.422, 8: 0.389
        // but cfg4 y 0.332 -> 0.345)
        if (MAXM * V >= 64) {
            for (int k = 0; k < bd.y; ++k) term(k);
        } else {
#pragma unroll 2
            for (int k = 0; k < bd.y; ++k) term(k);
        }
        if (CYC) {
            const int ns = __ldg(&T.Sn[set]);
            for (int k = 0; k < ns; ++k) {
                const int idx = __ldg(&T.Sidx[(size_t)set * T.Scap + k]);
                const double sv = __ldg(&T.Sval[(size_t)set * T.Scap + k]);
#pragma unroll
                for (int v = 0; v < V; ++v) sc[v] = fma(sv, rs[(idx * LPC + tx) * V + v], sc[v]);
            }
        }
    }
    // Eq.(8): x = xt - v yL - w yR (- q s for periodic lines), then store
#pragma unroll
    for (int jj = 0; jj < MAXM; ++jj) {
        const double2 vw = UNI ? make_double2(U.v[UNI ? jj * 6 + F_V : 0], U.v[UNI ? jj * 6 + F_W : 0]) : (TS ? trow[jj * 3 + 2] : __ldg(&rt[jj * 3 + 2]));     // {v, w}
        double qj = 0.0;
        if (CYC) qj = __ldg(reinterpret_cast<const double*>(&rt[jj * 3 + 0]) + 1);   // {l, q}
#pragma unroll
        for (int v = 0; v < V; ++v) {
            double r = fma(-vw.x, yL[v], x[jj][v]);
            r = fma(-vw.y, yR[v], r);
            if (CYC) r = fma(-qj, sc[v], r);
            x[jj][v] = r;
        }
        if (valid && (full || jj < m)) VecIO<V>::st(base + jj * rstride, x[jj]);
        if (MAXM * V > 8 && A.iface != nullptr && valid) {  // Alg.1 step 4 (slab sweeps): the interface rows, packed for the exchange
            double* ip = A.iface + ((long long)o * A.W + i) * V;
            if (p == 0 && jj == 0) VecIO<V>::st(ip, x[0]);
            if (p == P - 1 && jj == m - 1) VecIO<V>::st(ip + A.iface_plane, x[jj]);
        }
    }
    if (MAXM * V <= 8 && A.iface != nullptr && valid) {     // Alg.1 step 4 (slab sweeps): the interface rows, packed for the exchange.
        double* ip = A.iface + ((long long)o * A.W + i) * V;   // Tiny tiles: a chain of selects (the in-loop form below becomes a
        if (p == 0) VecIO<V>::st(ip, x[0]);                 // run-time index there, which puts the tile into local memory)
        if (p == P - 1) {
            double xlast[V];
#pragma unroll
            for (int v = 0; v < V; ++v) xlast[v] = x[0][v];
#pragma unroll
            for (int jj = 1; jj < MAXM; ++jj)
#pragma unroll
                for (int v = 0; v < V; ++v) xlast[v] = (jj < m) ? x[jj][v] : xlast[v];
            VecIO<V>::st(ip + A.iface_plane, xlast);
        }
    }
    if (xt + (int)gridDim.x < tiles_x) __syncthreads();     // rs is reused by the next tile
  }
}

// ---------------------------------------------------------------------------------------------------------
struct UnitArgs {
    double* data;
    long long nlines;
    int LPB;                 // whole lines per CTA
    int pad_en;              // pad the per-warp tile (partition length even)
    unsigned inv20;          // ceil(2^20 / q) for the pad index
};

template <int MAXM> constexpr int unit_block_threads() { return MAXM <= 8 ? 1024 : (MAXM <= 24 ? 512 : 256); }

template <int MAXM, bool UNI, bool CYC>
__global__ void __launch_bounds__(unit_block_threads<MAXM>())
k_unit(UnitArgs A, Tables T) {
    extern __shared__ double sm[];
    const int P = T.P, n = T.n;
    const int tl = threadIdx.x, lane = tl & 31, warp = tl >> 5;
    const int nthreads_real = A.LPB * P;
    const int nwarps = blockDim.x >> 5;
    constexpr int WT = 32 * MAXM + 48;                                 // per-warp tile capacity (doubles)
    double* tile = sm + (size_t)warp * WT;
    double* rf = sm + (size_t)nwarps * WT;                              // xt_first per thread
    double* rl = rf + blockDim.x;                                       // xt_last per thread

    const long long line0 = (long long)blockIdx.x * A.LPB;
    long long lines_here = A.nlines - line0; if (lines_here > A.LPB) lines_here = A.LPB;
    const int ll = tl / P, p = tl - ll * P;
    const bool valid = tl < nthreads_real && ll < lines_here;
    int pst = 0, m = 0;
    if (valid) sub_part(p, T.q, T.r, T.S, pst, m);
    const int cta_end = (int)lines_here * n;
    const int S = valid ? ll * n + pst : cta_end;                       // element offset in the CTA chunk
    const int e0 = __shfl_sync(0xffffffffu, S, 0);
    const int e1 = __shfl_sync(0xffffffffu, S + m, 31);
    const int count = e1 - e0;
    double* gptr = A.data + line0 * n + e0;
    auto padi = [&](int e) -> int { return A.pad_en ? e + (int)(((unsigned)e * A.inv20) >> 20) : e; };

    double x[MAXM];
#pragma unroll
    for (int k = 0; k < MAXM; ++k) { const int e = k * 32 + lane; x[k] = (e < count) ? __ldcs(gptr + e) : 0.0; }
#pragma unroll
    for (int k = 0; k < MAXM; ++k) { const int e = k * 32 + lane; if (e < count) tile[padi(e)] = x[k]; }
    __syncwarp();
    const int off = S - e0;
#pragma unroll
    for (int jj = 0; jj < MAXM; ++jj) x[jj] = (jj < m) ? tile[padi(off + jj)] : 0.0;

    // table access: UNI -> one table for every partition (warp-uniform), else per-partition columns (coalesced)
    const double* rows = T.rows;
    auto tab = [&](int jj, int f) -> double {
        if (UNI) return __ldg(rows + jj * 6 + f);
        return __ldg(rows + ((size_t)jj * 6 + f) * P + (valid ? p : 0));
    };
#pragma unroll
    for (int jj = 1; jj < MAXM; ++jj) x[jj] = fma(-tab(jj, F_L), x[jj - 1], x[jj]);
    x[MAXM - 1] *= tab(MAXM - 1, F_INV);
#pragma unroll
    for (int jj = MAXM - 2; jj >= 0; --jj) x[jj] = fma(-tab(jj, F_CP), x[jj + 1], x[jj] * tab(jj, F_INV));
    rf[tl] = x[0]; rl[tl] = x[MAXM - 1];                               // the plan's padding rows carry xt_last to slot MAXM-1 (a select
                                                                        // over jj == m-1 becomes a run-time index: the tile went to local memory)
    __syncthreads();
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
#pragma unroll
    for (int jj = 0; jj < MAXM; ++jj) {
        double r = fma(-tab(jj, F_V), yL, x[jj]);
        r = fma(-tab(jj, F_W), yR, r);
        if (CYC) r = fma(-tab(jj, F_Q), sc, r);
        if (jj < m) tile[padi(off + jj)] = r;
    }
    __syncwarp();
#pragma unroll
    for (int k = 0; k < MAXM; ++k) { const int e = k * 32 + lane; if (e < count) __stcs(gptr + e, tile[padi(e)]); }
}

// ---------------------------------------------------------------------------------------------------------
// THOMAS mode: one thread per line, in place in global memory (forward pass stores y, backward pass re-reads it).
// rows[(set*n + j)*6 + f].  cyc[set*4 + {0:g, 3:kappa}] for periodic lines.
template <int V, bool CYC>
__global__ void k_thomas_strided(StridedArgs A, const double* __restrict__ rows, const double* __restrict__ cyc, int n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.W) return;
    const int o = blockIdx.y;
    const int set = A.set_per_outer ? A.set0 + o : 0;
    double* base = A.data + ((long long)o * A.outer_stride + i) * V;
    const long long rstride = A.line_stride * V;
    const double* rt = rows + (size_t)set * n * 6;
    double prev[V], cur[V], dot[V];
#pragma unroll
    for (int v = 0; v < V; ++v) { prev[v] = 0.0; dot[v] = 0.0; }
    for (int j = 0; j < n; ++j) {
        const double l = __ldg(rt + (size_t)j * 6 + F_L);
        VecIO<V>::ld(base + j * rstride, cur);
        if (CYC) {                                           // z.d = y_0 + g y_{n-1} (k_cyclic_z): the closure's scalar, one pass early
            const double zj = __ldg(rt + (size_t)j * 6 + F_V);
#pragma unroll
            for (int v = 0; v < V; ++v) dot[v] = fma(zj, cur[v], dot[v]);
        }
#pragma unroll
        for (int v = 0; v < V; ++v) { cur[v] = fma(-l, prev[v], cur[v]); prev[v] = cur[v]; }
        VecIO<V>::st(base + j * rstride, cur);
    }
    double ylast[V], sc[V];
#pragma unroll
    for (int v = 0; v < V; ++v) { prev[v] = 0.0; sc[v] = CYC ? __ldg(cyc + set * 4 + 3) * dot[v] : 0.0; }
    for (int j = n - 1; j >= 0; --j) {
        const double inv = __ldg(rt + (size_t)j * 6 + F_INV), cp = __ldg(rt + (size_t)j * 6 + F_CP);
        VecIO<V>::ld(base + j * rstride, cur);
#pragma unroll
        for (int v = 0; v < V; ++v) { cur[v] = fma(-cp, prev[v], cur[v] * inv); prev[v] = cur[v]; if (j == n - 1) ylast[v] = cur[v]; }
        if (CYC) {                                           // x_j = y_j - q_j s (Sherman-Morrison, Eq.(3)); prev keeps y_j
            const double qj = __ldg(rt + (size_t)j * 6 + F_Q);
#pragma unroll
            for (int v = 0; v < V; ++v) cur[v] = fma(-qj, sc[v], cur[v]);
        }
        VecIO<V>::st(base + j * rstride, cur);
    }
    if (A.iface != nullptr && !CYC) {                       // slab sweeps: pack rows 0 and n-1 (prev = x_0, ylast = x_{n-1})
        double* ip = A.iface + ((long long)o * A.W + i) * V;
        VecIO<V>::st(ip, prev);
        VecIO<V>::st(ip + A.iface_plane, ylast);
    }
}

// THOMAS mode of the Helmholtz y-solves when the shift differs from line to line (lambda = kx2[i] + kz2[m], the paper's
// cosine-x / Fourier-z Poisson solve): no table can be shared, so the thread that owns complex
// line (i, m) factorises on the fly -- a_j = lo_j, c_j = up_j, b_j = -(a_j + c_j) - lambda, Neumann ends, lambda == 0
// pinned at j = 0 (L172) -- stores the scaled forward-eliminated right-hand side in place and the scaled
// super-diagonal c'_j in the workspace ws[m][j][i], and substitutes back.  Two passes over HBM: the GPU baseline.
__global__ void k_thomas_helm_lines(double2* __restrict__ data, double* __restrict__ ws, int nx, int ny,
                                    const double* __restrict__ lo, const double* __restrict__ up,
                                    const double* __restrict__ kx2, const double* __restrict__ kz2) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nx) return;
    const int m = blockIdx.y;
    const double lam = __dadd_rn(__ldg(kx2 + i), __ldg(kz2 + m));
    const bool pinned = lam == 0.0;
    double2* base = data + (size_t)m * ny * nx + i;
    double* wb = ws + (size_t)m * ny * nx + i;
    double cp = 0.0;
    double2 prev = make_double2(0.0, 0.0);
    for (int j = 0; j < ny; ++j) {
        double aj = __ldg(lo + j), cj = __ldg(up + j);
        double bj = __dsub_rn(-__dadd_rn(aj, cj), lam);
        if (j == 0) { bj = __dsub_rn(-cj, lam); aj = 0.0; }
        if (j == ny - 1) { bj = __dsub_rn(-aj, lam); cj = 0.0; }
        double2 d = base[(size_t)j * nx];
        if (pinned && j == 0) { bj = 1.0; cj = 0.0; d = make_double2(0.0, 0.0); }
        const double den = bj - aj * cp;                    // Thomas: c'_j = c_j/den, d'_j = (d_j - a_j d'_{j-1})/den
        cp = cj / den;
        prev.x = (d.x - aj * prev.x) / den;
        prev.y = (d.y - aj * prev.y) / den;
        base[(size_t)j * nx] = prev;
        wb[(size_t)j * nx] = cp;
    }
    double2 nxt = prev;                                      // x_{n-1} = d'_{n-1}
    for (int j = ny - 2; j >= 0; --j) {
        const double c1 = wb[(size_t)j * nx];
        double2 d = base[(size_t)j * nx];
        d.x = d.x - c1 * nxt.x; d.y = d.y - c1 * nxt.y;
        base[(size_t)j * nx] = d;
        nxt = d;
    }
}

// ---------------------------------------------------------------------------------------------------------
// PDD / PPT for the Helmholtz y-solves when every line has its own shift lambda = kx2[i] + kz2[m] (
// the paper's TDMA-C workload after the cosine-x and Fourier-z transforms).  Nothing is
// matrix-only any more, so the thread that owns (complex line, partition) does the whole of Eq.(5)-(6) on the fly:
//   forward  : pivots, c'_j, the scaled right-hand side (re, im) and the scaled left spike, one division per row;
//   backward : xt, the left spike v and the right spike w (w takes the slot of c'_j, which is dead by then);
// the interface values and spike ends go to shared memory; PDD solves its two 2x2 blocks per thread (Alg.1 step 5), PPT
// solves the block-tridiagonal Z in natural order (2x2 diagonal blocks [[1, w_last],[v_first, 1]]; DESIGN.md reading
// A7) by block parallel cyclic reduction over the line's P threads, ceil(log2(P-1)) steps of one division each;
// then Eq.(8).  RAG = false: n = P*M exactly.  RAG = true: the partition map of tdx_partition_bounds (q = n / P rows, the
// first rq = n % P partitions one more, all <= M); slots jj >= m of a partition are padding rows (a = -1, b = 1, c = 0,
// d = 0), which copy xt_last, v_last and w_last along to slot M-1 so that no register array is indexed at run time.
// HBM traffic: 32 B per complex point; lo/up/kx2/kz2 come from L1.
template <int M, bool RAG>
__global__ void __maxnreg__(M <= 8 ? 128 : (M <= 12 ? 168 : 208))
k_helm_lines(double2* __restrict__ data, int nx, int ny, int P, int q, int rq, int ppt, int pf,
             const double* __restrict__ lo, const double* __restrict__ up,
             const double* __restrict__ kx2, const double* __restrict__ kz2) {
    extern __shared__ double hs[];
    const int tx = threadIdx.x, p = threadIdx.y, LPC = blockDim.x;
    const int i = blockIdx.x * LPC + tx;
    const bool valid = i < nx;
    const int m = blockIdx.y;
    const double lam = valid ? __dadd_rn(__ldg(kx2 + i), __ldg(kz2 + m)) : 1.0;
    const bool pinned = lam == 0.0;
    const int start = RAG ? part_start(p, q, rq) : p * M;
    const int mr = RAG ? q + (p < rq ? 1 : 0) : M;                  // real rows of this partition
    double2* base = data + ((size_t)m * ny + start) * nx + i;
    // shared layout, all indexed [p][tx]: xf, xl (double2), vf, vl, wf, wl; PPT adds beta, idet, r0, r1 (double2 r)
    const int S = P * LPC;
    double2* s_xf = reinterpret_cast<double2*>(hs);
    double2* s_xl = s_xf + S;
    double* s_vf = reinterpret_cast<double*>(s_xl + S);
    double* s_vl = s_vf + S;
    double* s_wf = s_vl + S;
    double* s_wl = s_wf + S;
    double2* s_y0 = reinterpret_cast<double2*>(s_wl + S);          // (spare)
    double2* s_y1 = s_y0 + S;                                      // PPT: x_first_i; the PCR buffers follow it
    const int me = p * LPC + tx;

    double2 y[M];
    double f[M], cp[M];
#pragma unroll
    for (int jj = 0; jj < M; ++jj) y[jj] = (valid && (!RAG || jj < mr)) ? __ldcs(base + (size_t)jj * nx) : make_double2(0.0, 0.0);
    if (pf > 0 && (tx & 7) == 0) {                                   // L2 prefetch of the tile `pf` CTAs ahead, one lane per 128-byte line
        const long long lin = (long long)blockIdx.y * gridDim.x + blockIdx.x + pf;
        if (lin < (long long)gridDim.x * gridDim.y) {
            const int by = (int)(lin / gridDim.x), bx = (int)(lin - (long long)by * gridDim.x);
            if (bx * LPC + tx < nx) {
                const double2* pb = data + ((size_t)by * ny + start) * nx + bx * LPC + tx;
#pragma unroll
                for (int jj = 0; jj < M; ++jj) if (!RAG || jj < mr) asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + (size_t)jj * nx));
            }
        }
    }
    double wl = 0.0;
    {   // forward elimination of the block (a_first and c_last of the block are zeroed: Alg.1 step 2)
        double cprev = 0.0, fprev = 0.0;
        double2 yprev = make_double2(0.0, 0.0);
#pragma unroll
        for (int jj = 0; jj < M; ++jj) {
            const int j = start + jj;
            const bool pad = RAG && jj >= mr;
            double aj = -1.0, cj = 0.0, bj = 1.0;                    // padding row: y_jj = y_{jj-1}
            if (!pad) {
                aj = __ldg(lo + j); cj = __ldg(up + j);
                bj = __dsub_rn(-__dadd_rn(aj, cj), lam);
                if (j == 0) { bj = __dsub_rn(-cj, lam); aj = 0.0; }
                if (j == ny - 1) { bj = __dsub_rn(-aj, lam); cj = 0.0; }
                if (pinned && j == 0) { bj = 1.0; cj = 0.0; y[0] = make_double2(0.0, 0.0); }
            }
            const double ae = (jj == 0) ? 0.0 : aj, ce = (RAG ? jj >= mr - 1 : jj == M - 1) ? 0.0 : cj;
            const double inv = 1.0 / (bj - ae * cprev);
            cp[jj] = ce * inv;
            y[jj].x = (y[jj].x - ae * yprev.x) * inv;
            y[jj].y = (y[jj].y - ae * yprev.y) * inv;
            f[jj] = (jj == 0) ? aj * inv : -ae * fprev * inv;       // left spike: rhs a_first e_first
            if (RAG ? jj == mr - 1 : jj == M - 1) wl = cj * inv;     // right spike: rhs c_last e_last
            cprev = cp[jj]; fprev = f[jj]; yprev = y[jj];
        }
    }
    {   // backward substitution: xt, v, w (w overwrites c')
        double wn = wl;
        cp[M - 1] = wl;
#pragma unroll
        for (int jj = M - 2; jj >= 0; --jj) {
            const double c1 = cp[jj];
            y[jj].x = y[jj].x - c1 * y[jj + 1].x;
            y[jj].y = y[jj].y - c1 * y[jj + 1].y;
            f[jj] = f[jj] - c1 * f[jj + 1];
            wn = (RAG && jj >= mr - 1) ? wl : -c1 * wn;              // padding slots hold w_last
            cp[jj] = wn;
        }
    }
    s_xf[me] = y[0]; s_xl[me] = y[M - 1];
    s_vf[me] = f[0]; s_vl[me] = f[M - 1];
    s_wf[me] = cp[0]; s_wl[me] = cp[M - 1];
    __syncthreads();
    double2 yL = make_double2(0.0, 0.0), yR = make_double2(0.0, 0.0);
    if (!ppt) {
        // PDD: interface blocks [[1, w_last^(i-1)],[v_first^(i), 1]] only
        if (p >= 1) {
            const int lft = me - LPC;
            const double w = s_wl[lft], v = s_vf[me];
            const double idet = 1.0 / (1.0 - w * v);
            yL.x = (s_xl[lft].x - w * s_xf[me].x) * idet;
            yL.y = (s_xl[lft].y - w * s_xf[me].y) * idet;
        }
        if (p <= P - 2) {
            const int rgt = me + LPC;
            const double w = s_wl[me], v = s_vf[rgt];
            const double idet = 1.0 / (1.0 - w * v);
            yR.x = (s_xf[rgt].x - v * s_xl[me].x) * idet;
            yR.y = (s_xf[rgt].y - v * s_xl[me].y) * idet;
        }
    } else {
        // PPT (L126-146, L156): the reduced system Z in natural order, unknown block i = (s_i, t_i) =
        // (x_last_{i-1}, x_first_i), i = 1..K, K = P-1:
        //   row A_i: l_i s_{i-1} + s_i + beta_i t_i = r0_i      l_i = v_last^(i-1), beta_i = w_last^(i-1)
        //   row B_i: gamma_i s_i + t_i + u_i t_{i+1} = r1_i     gamma_i = v_first^(i), u_i = w_first^(i)
        // i.e. block tridiagonal with D_i = [[1, beta_i],[gamma_i, 1]] and rank-one couplings L_i = l_i e0 e0^T,
        // U_i = u_i e1 e1^T.  Solved by block parallel cyclic reduction across the line's P threads (thread p owns block
        // p): a step of distance d substitutes blocks i-d and i+d into block i,
        //   beta_i += l_i u_{i-d} e01_{i-d},  r0_i -= l_i (D^-1 r)_{i-d,0},  l_i <- -l_i l_{i-d} idet_{i-d},
        //   gamma_i += u_i l_{i+d} e10_{i+d}, r1_i -= u_i (D^-1 r)_{i+d,1},  u_i <- -u_i u_{i+d} idet_{i+d},
        // (idet = 1/(1 - beta gamma), e01 = beta idet, e10 = gamma idet) which keeps the form of D, L and U; after
        // ceil(log2 K) steps the blocks are decoupled and (s_i, t_i) = D_i^-1 r_i.  No pivoting is needed in this order
        // (unit diagonal, |spikes| < 1; reading A7 -- the permuted Z-bar of Eq.(10) would need it).
        const int K = P - 1;
        double beta = 0.0, gamma = 0.0, l = 0.0, u = 0.0;
        double2 r0 = make_double2(0.0, 0.0), r1 = make_double2(0.0, 0.0);
        if (p >= 1) {
            const int a = me - LPC;                                  // partition p-1
            beta = s_wl[a]; gamma = s_vf[me];
            l = (p >= 2) ? s_vl[a] : 0.0;
            u = (p <= K - 1) ? s_wf[me] : 0.0;
            r0 = s_xl[a]; r1 = s_xf[me];
        }
        // Per step a block hands its neighbours products, not raw coefficients: to the block d to its right {u e01, l idet} and
        // q0, to the block d to its left {l e10, u idet} and q1 -- 16-byte pairs, 4 stores and 4 loads per step.
        double2* pc = s_y1 + S;                                      // 2 buffers x {cR, q0, cL, q1} x S (16 bytes each)
        int buf = 0;
        double2 q0, q1;
        for (int d = 1;; d <<= 1) {
            const double idet = 1.0 / (1.0 - beta * gamma);
            q0 = make_double2((r0.x - beta * r1.x) * idet, (r0.y - beta * r1.y) * idet);
            q1 = make_double2((r1.x - gamma * r0.x) * idet, (r1.y - gamma * r0.y) * idet);
            if (d >= K) break;                                       // uniform over the CTA
            double2* B = pc + buf * 4 * S + me;
            B[0] = make_double2(u * beta * idet, l * idet); B[S] = q0;
            B[2 * S] = make_double2(l * gamma * idet, u * idet); B[3 * S] = q1;
            // couplings below 1e-30 of the unit diagonal are invisible in fp64: once every block of the CTA's lines is
            // decoupled (decayed spikes: high wavenumbers away from the wall) the remaining steps would change nothing
            if (!__syncthreads_or(fabs(l) > 1e-30 || fabs(u) > 1e-30)) break;
            if (p >= 1) {
                double ln = 0.0, un = 0.0;
                const int off = d * LPC;
                if (p - d >= 1) {
                    const double2 cR = B[-off], qL = B[S - off];
                    beta = fma(l, cR.x, beta);
                    r0.x = fma(-l, qL.x, r0.x); r0.y = fma(-l, qL.y, r0.y);
                    ln = -l * cR.y;
                }
                if (p + d <= K) {
                    const double2 cL = B[2 * S + off], qR = B[3 * S + off];
                    gamma = fma(u, cL.x, gamma);
                    r1.x = fma(-u, qR.x, r1.x); r1.y = fma(-u, qR.y, r1.y);
                    un = -u * cL.y;
                }
                l = ln; u = un;
            }
            buf ^= 1;
        }
        s_y1[me] = q1;                                               // t_p = x_first_p
        __syncthreads();
        if (p >= 1) yL = q0;                                         // s_p = x_last_{p-1}
        if (p <= P - 2) yR = s_y1[me + LPC];                         // t_{p+1} = x_first_{p+1}
    }
    // Eq.(8): x = xt - v yL - w yR
#pragma unroll
    for (int jj = 0; jj < M; ++jj) {
        double2 r = y[jj];
        r.x = fma(-f[jj], yL.x, r.x); r.y = fma(-f[jj], yL.y, r.y);
        r.x = fma(-cp[jj], yR.x, r.x); r.y = fma(-cp[jj], yR.y, r.y);
        if (valid && (!RAG || jj < mr)) __stcs(base + (size_t)jj * nx, r);
    }
}

// THOMAS mode along x, warp-tiled: a warp owns 32 consecutive lines and walks them 32 columns at a time.  The 32 x 32 tile comes
// in with coalesced 256-byte row reads (lane = column), is turned through shared memory (33-double rows: conflict-free both
// ways) so that lane = line runs its recurrence over the 32 columns, and goes back the same way -- forward pass up the line,
// backward pass down (periodic lines: the closure's scalar s comes out of the forward pass, k_cyclic_z).  The
// one-thread-per-line form it replaces read 8 useful bytes per 32-byte sector (cfg5 10.8 ms against 3.1 ms for the strided
// directions); this one moves the same 32 B per value with full sectors.  Shared memory: 32 * 33 doubles per warp.
template <bool CYC>
__global__ void __launch_bounds__(128) k_thomas_unit_tiled(double* __restrict__ data, long long nlines, const double* __restrict__ rows,
                                                          const double* __restrict__ cyc, int n) {
    extern __shared__ double tt[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double* tile = tt + w * (32 * 33);
    const long long line0 = ((long long)blockIdx.x * (blockDim.x >> 5) + w) * 32;
    if (line0 >= nlines) return;
    const int nl = (int)min((long long)32, nlines - line0);
    double* base = data + line0 * n;
    // the tile of the NEXT step is in flight (32 loads per lane, in registers) while the current one is computed
    double nxt[32];
    auto fetch = [&](int c0) {
        const bool in = c0 >= 0 && c0 + lane < n;
#pragma unroll
        for (int r = 0; r < 32; ++r) nxt[r] = (in && r < nl) ? base[(long long)r * n + c0 + lane] : 0.0;
    };
    auto land = [&]() {
#pragma unroll
        for (int r = 0; r < 32; ++r) tile[r * 33 + lane] = nxt[r];
    };
    auto put = [&](int c0) {
        if (c0 + lane < n) {
#pragma unroll
            for (int r = 0; r < 32; ++r) if (r < nl) base[(long long)r * n + c0 + lane] = tile[r * 33 + lane];
        }
    };
    double prev = 0.0, dot = 0.0;
    fetch(0);
    for (int c0 = 0; c0 < n; c0 += 32) {                            // forward: y_j = d_j - l_j y_{j-1}
        const int nc = min(32, n - c0);
        land();
        fetch(c0 + 32 < n ? c0 + 32 : -1);
        __syncwarp();
        if (lane < nl) {
#pragma unroll 8
            for (int k = 0; k < nc; ++k) {
                const double dj = tile[lane * 33 + k];
                if (CYC) dot = fma(__ldg(rows + (size_t)(c0 + k) * 6 + F_V), dj, dot);      // z.d (k_cyclic_z)
                const double cur = fma(-__ldg(rows + (size_t)(c0 + k) * 6 + F_L), prev, dj);
                tile[lane * 33 + k] = cur; prev = cur;
            }
        }
        __syncwarp();
        put(c0);
        __syncwarp();
    }
    prev = 0.0;
    const double sc = CYC ? __ldg(cyc + 3) * dot : 0.0;               // s = kappa (y_0 + g y_{n-1}) = kappa z.d of this lane's line
    const int clast = ((n - 1) / 32) * 32;
    // The backward pass re-reads what the forward pass has just written through this same warp: ordinary loads after the
    // stores of the same thread are ordered, and a lane only reads columns it wrote itself (lane = column in both).
    fetch(clast);
    for (int c0 = clast; c0 >= 0; c0 -= 32) {                        // backward: x_j = y_j inv_j - c'_j x_{j+1}
        const int nc = min(32, n - c0);
        land();
        fetch(c0 - 32);
        __syncwarp();
        if (lane < nl) {
#pragma unroll 8
            for (int k = nc - 1; k >= 0; --k) {
                const int j = c0 + k;
                const double cur = fma(-__ldg(rows + (size_t)j * 6 + F_CP), prev, tile[lane * 33 + k] * __ldg(rows + (size_t)j * 6 + F_INV));
                prev = cur;                                                                      // y_j; x_j = y_j - q_j s (Eq.(3))
                tile[lane * 33 + k] = CYC ? fma(-__ldg(rows + (size_t)j * 6 + F_Q), sc, cur) : cur;
            }
        }
        __syncwarp();
        put(c0);
        __syncwarp();
    }
}

}  // namespace tdx
