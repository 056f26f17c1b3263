// tdx_slab.cuh -- the paper's own decomposition one level up ("the computational domain is divided in the
// wall-normal direction", Algorithm 1, PPT across GPUs L156/L174): every GPU (rank) owns a slab
// of n_loc consecutive rows of each line of the slab direction and is ONE partition of the PDD / PPT method.
//
//   Alg.1 step 2-3   cut the couplings at the slab ends and solve A_r xt = d locally: the slab's own sweep kernels
//                    (tdx_kernels.cuh / tdx_tma.cuh) with the cut operator as a user-coefficient plan; the spikes
//                    A_r v = a_first e_first, A_r w = c_last e_last are matrix-only, so they are plan-time vectors here
//                    (k_slab_spikes) instead of two extra right-hand sides per line (R(9M), L228-231).
//   step 4 / 6       the interface rows xt_first, xt_last of the slab are packed into one buffer BY THE SWEEP KERNEL's own
//                    store loop (StridedArgs::iface: iface[0][outer][inner] = row 0, iface[1][..] = row n_loc-1) that the
//                    caller exchanges: neighbour send/recv for PDD (L244-256), one all-gather for PPT (L156, L174).
//   step 5 + 7       k_slab_correct: per line, the interface unknowns (PDD: the two 2x2 blocks of L148-154; PPT: two rows
//                    of the plan-time Z^-1 of the rank-level reduced system, Eq.(7)) in the prologue, then
//                    x = xt - v yL - w yR (Eq.(8)) over the slab.
// One launch per phase: the messages are 2 / n_loc of the slab, so launch and exchange latency is what a sweep pays for
// beyond its two passes.  The correction is a second pass over the slab (8 B read + 8 B written per value), as step 7 is in
// the paper.
#pragma once
#include <cuda_runtime.h>

namespace tdx {

// One thread per rank r: spikes of the block rows [starts[r], starts[r+1]) of the global operator (a, b, c), couplings
// at the block ends cut.  ends[r*4 + {0: v_first, 1: v_last, 2: w_first, 3: w_last}]; rank `me` also writes its whole
// v and w (n_loc doubles each).  scratch: nranks * 3 * nmax doubles.  Rank 0 has no left spike, rank R-1 no right one.
__global__ void k_slab_spikes(int R, const int* __restrict__ starts, const double* __restrict__ a, const double* __restrict__ b,
                              const double* __restrict__ c, int me, int nmax, double* __restrict__ scratch,
                              double* __restrict__ ends, double* __restrict__ v_out, double* __restrict__ w_out) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    const int s = starts[r], e = starts[r + 1], n = e - s;
    double* cp = scratch + (size_t)r * 3 * nmax;
    double* v = cp + nmax;
    double* w = v + nmax;
    double cprev = 0.0, vprev = 0.0, wprev = 0.0;
    for (int jj = 0; jj < n; ++jj) {
        const int j = s + jj;
        const double ae = (jj == 0) ? 0.0 : a[j], ce = (jj == n - 1) ? 0.0 : c[j];
        const double inv = 1.0 / (b[j] - ae * cprev);
        const double rv = (jj == 0 && r >= 1) ? a[j] : 0.0;
        const double rw = (jj == n - 1 && r <= R - 2) ? c[j] : 0.0;
        cp[jj] = ce * inv;
        v[jj] = (rv - ae * vprev) * inv;
        w[jj] = (rw - ae * wprev) * inv;
        cprev = cp[jj]; vprev = v[jj]; wprev = w[jj];
    }
    for (int jj = n - 2; jj >= 0; --jj) {
        v[jj] -= cp[jj] * v[jj + 1];
        w[jj] -= cp[jj] * w[jj + 1];
    }
    ends[r * 4 + 0] = v[0]; ends[r * 4 + 1] = v[n - 1]; ends[r * 4 + 2] = w[0]; ends[r * 4 + 3] = w[n - 1];
    if (r == me) for (int jj = 0; jj < n; ++jj) { v_out[jj] = v[jj]; w_out[jj] = w[jj]; }
}

// Alg.1 steps 5 and 7 in ONE pass over the slab [outer][n_loc][inner].  Thread = two adjacent inner elements (inner is
// even) of one outer index.  Prologue (step 5 / Eq.(7)): the two interface unknowns of the thread's lines, yL = x_last of
// rank-1, yR = x_first of rank+1 (zero where there is no neighbour) --
//   PDD: the two 2x2 blocks of L148-154, coef = {wl_prev, vf_me, wl_me, vf_next};
//   PPT: two rows of the plan-time Z^-1 of the rank-level reduced system, coef[k] (yL) and coef[K + k] (yR), K = 2(R-1).
// own: [2][plane] of this rank (xt_first, xt_last); nbr: PDD [2][plane] = (xt_last of rank-1, xt_first of rank+1); PPT
// [R][2][plane] gathered from every rank.  Then Eq.(8) (step 7): x = xt - v yL - w yR, marching over rows [j0, j1) of the
// slab; grid.y slices the rows only when the plane alone has too few threads to fill the GPU (each slice then repeats the
// prologue, which reads 4 (PDD) or 2R (PPT) plane values against 2 JT slab values).
template <bool PPT>
__global__ void __launch_bounds__(128) k_slab_correct(double* __restrict__ field, const double* __restrict__ own, const double* __restrict__ nbr,
                                                      const double* __restrict__ coef, const double* __restrict__ v, const double* __restrict__ w,
                                                      int rank, int R, int n_loc, long long inner, long long outer, int JT) {
    const long long plane = inner * outer;
    const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 2;
    if (i >= inner) return;
    const long long o = blockIdx.z;
    const long long q = o * inner + i;
    double2 yL = make_double2(0.0, 0.0), yR = make_double2(0.0, 0.0);
    if (!PPT) {
        const double2 xf = *reinterpret_cast<const double2*>(own + q), xl = *reinterpret_cast<const double2*>(own + plane + q);
        if (rank >= 1) {
            const double wl = coef[0], vf = coef[1], idet = 1.0 / (1.0 - wl * vf);
            const double2 pl = *reinterpret_cast<const double2*>(nbr + q);                 // xt_last of rank-1
            yL = make_double2((pl.x - wl * xf.x) * idet, (pl.y - wl * xf.y) * idet);
        }
        if (rank <= R - 2) {
            const double wl = coef[2], vf = coef[3], idet = 1.0 / (1.0 - wl * vf);
            const double2 nf = *reinterpret_cast<const double2*>(nbr + plane + q);         // xt_first of rank+1
            yR = make_double2((nf.x - vf * xl.x) * idet, (nf.y - vf * xl.y) * idet);
        }
    } else {
        const int K = 2 * (R - 1);
        for (int ib = 1; ib <= R - 1; ++ib) {                        // reduced right-hand side: (xt_last^(ib-1), xt_first^(ib))
            const double2 r0 = *reinterpret_cast<const double2*>(nbr + ((size_t)(ib - 1) * 2 + 1) * plane + q);
            const double2 r1 = *reinterpret_cast<const double2*>(nbr + ((size_t)ib * 2 + 0) * plane + q);
            const double gl0 = coef[2 * ib - 2], gl1 = coef[2 * ib - 1], gr0 = coef[K + 2 * ib - 2], gr1 = coef[K + 2 * ib - 1];
            yL.x += gl0 * r0.x + gl1 * r1.x; yL.y += gl0 * r0.y + gl1 * r1.y;
            yR.x += gr0 * r0.x + gr1 * r1.x; yR.y += gr0 * r0.y + gr1 * r1.y;
        }
    }
    const int j0 = blockIdx.y * JT, j1 = min(n_loc, j0 + JT);
    double* p = field + (o * n_loc + j0) * inner + i;
#pragma unroll 4
    for (int j = j0; j < j1; ++j, p += inner) {
        double2 x = __ldcs(reinterpret_cast<const double2*>(p));
        const double vj = __ldg(v + j), wj = __ldg(w + j);
        x.x = fma(-vj, yL.x, x.x); x.y = fma(-vj, yL.y, x.y);
        x.x = fma(-wj, yR.x, x.x); x.y = fma(-wj, yR.y, x.y);
        __stcs(reinterpret_cast<double2*>(p), x);
    }
}

}  // namespace tdx
