// tdx_general.cuh -- batched tridiagonal solve with PER-LINE coefficients and diagonal pivoting.
// for the y-solves of the Poisson equation "a parallel tridiagonal solver with diagonal pivoting is used
// [3]" because those systems are only weakly dominant (L172).  This is that role for systems that are not dominant at
// all: every line brings its own a, b, c (three more field-sized arrays, +24 B per value -- SURVEY 8(d) counts it), and
// the elimination chooses 1x1 or 2x2 diagonal pivots without row interchanges (the criterion of the diagonal-pivoting
// family [3] builds on: with sigma = max(|c_i|, |a_{i+1}|, |b_{i+1}|, |c_{i+1}|, |a_{i+2}|) take the 1x1 pivot b_i when
// |b_i| sigma >= kappa |c_i a_{i+1}|, kappa = (sqrt 5 - 1)/2, else the 2x2 block of rows i, i+1).
//
// Two kernels: k_general_part, the partition method (Eq.(5)-(8) per line with pivoted local solves, one pass over HBM),
// and k_general_lines, one thread per line over the whole line (two passes: the robust path the partition kernel hands
// numerically singular blocks to, the baseline it is measured against, and the periodic variant).  In k_general_lines all
// lanes of a warp walk the rows in lockstep -- a lane whose row is the second row of a 2x2 pivot idles for that row -- so a
// rolling three-row window in registers loads every coefficient exactly once.
#pragma once
#include <cuda_runtime.h>
#include "tdx_plan.cuh"

namespace tdx {

// ---------------------------------------------------------------------------------------------------------------------
// The partition method with per-line coefficients and diagonal pivoting inside the partitions: ONE pass over HBM,
// 32 B read (a, b, c, d) + 8 B written per value (16 + 24 B per value).
//
// Thread = (line, partition of <= M rows).  The thread keeps its rows of a, b, c, d in registers and runs Eq.(5)-(6) on
// the fly -- the block A_p with its end couplings cut (Alg.1 step 2), eliminated with 1x1 / 2x2 diagonal pivots (same
// criterion as k_general_forward), for three right-hand sides at once: d, the left spike a_first e_first and the right
// spike c_last e_last -- then the reduced system of the line (Eq.(7); natural order, 2x2 diagonal blocks, block parallel
// cyclic reduction over the line's P threads exactly as in k_helm_lines) and the correction Eq.(8).
//
// A partition method needs every block A_p (and the reduced system, solved here without pivoting) to be numerically
// regular, which a regular line does not guarantee: the solver [3] the paper uses has the same premise.  So the result
// is CHECKED before it is stored: every thread evaluates the line's equations in its rows (the coefficients once more,
// the neighbours' actual end values through shared memory) and ONE row whose componentwise backward error exceeds
// kGeneralBackwardError makes the whole line fall back: nothing of it is stored, its index goes to a list, and
// k_general_lines afterwards solves the listed lines one thread per line with diagonal pivoting over the whole line (two
// passes, workspace).  What is stored therefore has the backward error of a stable elimination, whatever the blocks were
// like.  On weakly dominant systems (the paper's Poisson y-systems, L172-174) no line falls back; on random non-dominant
// ones many do.
//
// Addressing: element (outer o, line l, row j) = o * outer_stride + l * lane_stride + j * row_stride.  STRIDED (y, z lines):
// lanes of a warp = adjacent lines (lane_stride 1: coalesced 8-byte lanes); UNIT (x lines): lanes = adjacent partitions of
// one line (row_stride 1: a warp reads one contiguous piece of memory, 8 rows per lane, through L1).
struct GeneralArgs {
    const double *a, *b, *c;
    double* d;
    int n, P, q, r;                      // partition map of tdx_partition_bounds(n, P)
    long long W, lane_stride, row_stride, outer_stride;
    int periodic;                        // not used by the partition kernel (periodic lines take the two-pass path)
    unsigned int* fb_count;              // number of lines that fell back
    unsigned int* fb_lines;              // their indices o * W + l
    unsigned int fb_cap;
    unsigned char* fb_flag;              // the same lines as one byte per line (1 = fell back): for the dense case, see k_general_lines
    // method choice on the device (default method of a pivoting solve along y / z, tdx.cu): sel[0] = rows of k_general_sample's
    // sample that are not diagonally dominant.  More than a quarter of nsamp: the optimistic partition pass would be wasted
    // work (most lines would be re-solved), so the kernels of the PARTITION method return at once and the all-lines launch of
    // k_general_lines (sel_lines = 1) does the work; else the other way round.  sel = NULL: no choice, every kernel runs.
    const unsigned int* sel;
    unsigned int nsamp;
    int sel_lines;
};

__device__ __forceinline__ bool general_deselected(const GeneralArgs& G) {
    if (G.sel == nullptr) return false;
    const bool lines = __ldg(G.sel) * 4u > G.nsamp;
    return lines != (G.sel_lines != 0);
}

// The sample: nsamp rows spread over the whole field (a multiplicative hash of the thread index), counted when
// |b| < |a| + |c|.  One launch of a few microseconds; the count is final when the kernels behind it on the stream start.
__global__ void k_general_sample(const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ c,
                                 unsigned long long npts, unsigned int nsamp, unsigned int* __restrict__ count) {
    const unsigned int t = blockIdx.x * blockDim.x + threadIdx.x;
    bool nd = false;
    if (t < nsamp) {
        const unsigned long long e = ((unsigned long long)t * 0x9E3779B97F4A7C15ull >> 11) % npts;
        nd = !(fabs(__ldg(b + e)) >= fabs(__ldg(a + e)) + fabs(__ldg(c + e)));
    }
    const unsigned m = __ballot_sync(0xffffffffu, nd);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(count, (unsigned)__popc(m));
}

// A line is accepted when every block was "tame" (1x1 pivots only, spikes <= 1: what a diagonally dominant block does -- the
// partition method is stable there, and a nearly singular dominant line, eps ~ 1e-6, cannot meet a backward-error test:
// its reduced system is as ill-conditioned as the line), or else when the componentwise backward error of what was computed,
// max_j |a_j x_{j-1} + b_j x_j + c_j x_{j+1} - d_j| / (|a_j x_{j-1}| + |b_j x_j| + |c_j x_{j+1}| + |d_j|), stays below this
// (a few roundings of a stable elimination; the forward error is then within cond(A) times it, whatever happened inside)
// Register budgets (measured on cfg5): pivoted blocks 128; plain elimination 96 for strided lines (two CTAs of
// 8 lines x 36 partitions per SM: y 8.0 -> 7.05 ms against 112 / 128 registers) and 112 for x lines (one 512-thread CTA either way).
constexpr double kGeneralBackwardError = 128.0 * 2.220446049250313e-16;

// FULL: every partition has exactly M rows (n = P * M): the ragged-partition selects and padding rows compile away.
// PIVOT = false is also the OPTIMISTIC first pass of a pivoting solve (tdx.cu): plain elimination, and a block counts as
// tame only if its LU factors are componentwise stable -- |L||U| <= 4|A|, which for a tridiagonal block is one test per row,
// |m_j c_{j-1}| + |b'_j| <= 4 |b_j| (the off-diagonal entries of |L||U| equal those of |A|; row- or column-dominant rows give
// <= 3) -- and its spikes stay <= 1; everything else must pass the backward-error test or goes to the pivoted per-line kernel.
template <int M, bool PIVOT, bool UNIT, bool FULL>
__global__ void __maxnreg__(M <= 8 ? (PIVOT ? 128 : (UNIT ? 112 : 96)) : 168)
k_general_part(GeneralArgs G) {
    if (general_deselected(G)) return;
    extern __shared__ double gs[];
    const int P = G.P;
    const int p = UNIT ? threadIdx.x : threadIdx.y, lt = UNIT ? threadIdx.y : threadIdx.x;
    const int L = UNIT ? blockDim.y : blockDim.x;                       // lines per CTA
    const int me = UNIT ? lt * P + p : p * L + lt, pst = UNIT ? 1 : L;   // shared-memory slot, distance to the next partition's slot
    const int S = P * L;
    const long long l = (long long)blockIdx.x * L + lt;
    const bool valid = l < G.W;
    const int o = blockIdx.y;
    const int start = FULL ? p * M : part_start(p, G.q, G.r), m = FULL ? M : G.q + (p < G.r ? 1 : 0);
    const long long e0 = (long long)o * G.outer_stride + (valid ? l : 0) * G.lane_stride + (long long)start * G.row_stride;
    const double kappa = 0.6180339887498949;

    // Rows jj >= m of a short partition are padding rows (-x_{jj-1} + x_jj = 0), which carry xt_last, v_last and w_last along to
    // slot M-1, so that no register array is ever indexed with a run-time row number (k_helm_lines does the same).
    // Alg.1 step 2: the couplings at the partition's ends are cut; they are the right-hand sides of the spikes (Eq.(6)).
    double A_[M], B_[M], C_[M], D_[M], F_[M];
    double clast = 0.0;
    {
        const double *pa = G.a + e0, *pb = G.b + e0, *pcc = G.c + e0, *pd = G.d + e0;
        const long long rs = G.row_stride;
        double av[M], cv[M];
#pragma unroll
        for (int jj = 0; jj < M; ++jj) {                                // all loads first: 4 M independent requests in flight
            const bool ld = valid && jj < m;
            av[jj] = ld ? __ldg(pa) : 0.0; B_[jj] = ld ? __ldg(pb) : 1.0; cv[jj] = ld ? __ldg(pcc) : 0.0; D_[jj] = ld ? __ldg(pd) : 0.0;
            pa += rs; pb += rs; pcc += rs; pd += rs;
        }
#pragma unroll
        for (int jj = 0; jj < M; ++jj) {
            const bool real = jj < m;
            A_[jj] = real ? (jj == 0 ? 0.0 : av[jj]) : -1.0;
            C_[jj] = (jj < m - 1) ? cv[jj] : 0.0;
            F_[jj] = (jj == 0 && p > 0) ? av[jj] : 0.0;
            if (jj == m - 1 && p < P - 1) clast = cv[jj];
        }
    }

    // forward elimination with 1x1 / 2x2 diagonal pivots; fl: 2 bits per row (0: 1x1, 1: first row of a 2x2 pivot, 2: second).
    // A row with a 1x1 pivot keeps the RECIPROCAL of its pivot in B_ (one division per row serves both passes).
    // The right spike's right-hand side c_last e_last enters in the backward pass (nothing precedes it to eliminate) -- but the
    // padding rows behind the last real row must carry w_last like xt_last and v_last: wpad = what the elimination of row
    // m-1 hands to row m.  Where no lane of the warp starts a 2x2 pivot the whole warp skips that code (warp-uniform branch).
    unsigned fl = 0;
    bool second = false, wild = false;
    double wpad = 0.0;
#pragma unroll
    for (int jj = 0; jj < M - 1; ++jj) {
        const double b0 = B_[jj], c0 = C_[jj], a1 = A_[jj + 1], b1 = B_[jj + 1];
        bool one = true;
        if (PIVOT) {
            const double c1 = C_[jj + 1], a2 = (jj + 2 < M) ? A_[jj + 2] : 0.0;
            const double sigma = fmax(fmax(fabs(c0), fabs(a1)), fmax(fabs(b1), fmax(fabs(c1), fabs(a2))));
            one = fabs(b0) * sigma >= kappa * fabs(c0 * a1);
        }
        const bool start2 = !second && !one;
        if (second) {                                                   // second row of a 2x2 pivot: nothing to eliminate with
            fl |= 2u << (2 * jj); second = false;
        } else if (one) {
            const double ib = 1.0 / b0, mlt = a1 * ib;
            B_[jj] = ib;
            B_[jj + 1] = fma(-mlt, c0, b1);
            // componentwise stability of the plain LU: |L||U| <= 4|A| (off the diagonal |L||U| = |A| exactly; NaN counts as wild)
            if (!PIVOT && !(fabs(mlt * c0) + fabs(B_[jj + 1]) <= 4.0 * fabs(b1))) wild = true;
            D_[jj + 1] = fma(-mlt, D_[jj], D_[jj + 1]);
            F_[jj + 1] = fma(-mlt, F_[jj], F_[jj + 1]);
            if (jj == m - 1) wpad = clast * ib;
        }
        if (PIVOT && __any_sync(0xffffffffu, start2)) {
            if (start2) {
                fl |= 1u << (2 * jj); second = true;
                const double idet = 1.0 / (b0 * b1 - a1 * c0);
                if (jj + 1 == m - 1) wpad = b0 * clast * idet;
                if (jj + 2 < M) {
                    const double c1 = C_[jj + 1], t = A_[jj + 2] * idet;
                    B_[jj + 2] = fma(-t, b0 * c1, B_[jj + 2]);
                    D_[jj + 2] = fma(-t, b0 * D_[jj + 1] - a1 * D_[jj], D_[jj + 2]);
                    F_[jj + 2] = fma(-t, b0 * F_[jj + 1] - a1 * F_[jj], F_[jj + 2]);
                }
            }
        }
    }
    if (second) fl |= 2u << (2 * (M - 1)); else B_[M - 1] = 1.0 / B_[M - 1];
    // backward substitution for xt (into D_), v (into F_) and w (into A_, whose entries are dead once their row is done)
    double growth = 0.0;
    {
        double xn = 0.0, vn = 0.0, wn = 0.0, px = 0.0, pv = 0.0, pw = 0.0;
#pragma unroll
        for (int jj = M - 1; jj >= 0; --jj) {
            const unsigned f = (fl >> (2 * jj)) & 3u;
            const double wr = (jj == m - 1) ? clast : (jj >= m ? wpad : 0.0);   // right spike: c_last e_last (+ what the padding rows carry)
            double x, v, w;
            if (!PIVOT || __all_sync(0xffffffffu, f == 0)) {
                const double ib = B_[jj], cj = C_[jj];
                x = (D_[jj] - cj * xn) * ib; v = (F_[jj] - cj * vn) * ib; w = (wr - cj * wn) * ib;
            } else if (f == 0) {
                const double ib = B_[jj], cj = C_[jj];
                x = (D_[jj] - cj * xn) * ib; v = (F_[jj] - cj * vn) * ib; w = (wr - cj * wn) * ib;
            } else if (f == 2) {                                        // rows jj-1, jj: [[b0, c0],[a1, b1]]
                constexpr int jm = 0;                                    // f == 2 never occurs at jj = 0
                const double b0 = B_[jj > 0 ? jj - 1 : jm], c0 = C_[jj > 0 ? jj - 1 : jm], a1 = A_[jj], b1 = B_[jj], cj = C_[jj];
                const double idet = 1.0 / (b0 * b1 - a1 * c0);
                const double r1x = D_[jj > 0 ? jj - 1 : jm], r2x = D_[jj] - cj * xn;
                const double r1v = F_[jj > 0 ? jj - 1 : jm], r2v = F_[jj] - cj * vn;
                const double r2w = wr - cj * wn;                        // the spike's right-hand side is zero in row jj-1
                x = (b0 * r2x - a1 * r1x) * idet; px = (b1 * r1x - c0 * r2x) * idet;
                v = (b0 * r2v - a1 * r1v) * idet; pv = (b1 * r1v - c0 * r2v) * idet;
                w = (b0 * r2w) * idet;            pw = (-c0 * r2w) * idet;
            } else { x = px; v = pv; w = pw; }
            D_[jj] = x; F_[jj] = v; A_[jj] = w;
            xn = x; vn = v; wn = w;
            growth = fmax(growth, fmax(fabs(v), fabs(w)));
        }
    }
    // A block that behaved like a diagonally dominant one -- 1x1 pivots only, spikes not above 1 (the
    // paper's systems) -- is the case the partition method is stable for: its lines are accepted as they are.
    const bool tame = (fl == 0u) && !wild && (growth <= 1.0 + 1e-9);
    const double xl = D_[M - 1], vl = F_[M - 1], wl = A_[M - 1];        // padding rows carried the last real row here
    const double xf = D_[0], vf = F_[0], wf = A_[0];

    // shared memory, all indexed [me]: xf, xl, vf, vl, wf, wl, t (x_first after the solve), 2 PCR buffers x 6, flags
    double* s_xf = gs;            double* s_xl = s_xf + S;  double* s_vf = s_xl + S;  double* s_vl = s_vf + S;
    double* s_wf = s_vl + S;      double* s_wl = s_wf + S;  double* s_t = s_wl + S;   double* pc = s_t + S;
    int* s_bad = reinterpret_cast<int*>(pc + 12 * S);           // per line of the CTA: [lt] a row failed the test, [L + lt] a block was not tame
    if (p == 0) { s_bad[lt] = 0; s_bad[L + lt] = 0; }
    s_xf[me] = xf; s_xl[me] = xl; s_vf[me] = vf; s_vl[me] = vl; s_wf[me] = wf; s_wl[me] = wl;
    __syncthreads();
    // Eq.(7): block i = (s_i, t_i) = (x_last_{i-1}, x_first_i), i = 1..P-1, owned by thread p = i (k_helm_lines has the derivation)
    const int K = P - 1;
    double beta = 0.0, gamma = 0.0, lo_ = 0.0, up_ = 0.0, r0 = 0.0, r1 = 0.0;
    if (p >= 1) {
        const int pa = me - pst;
        beta = s_wl[pa]; gamma = s_vf[me];
        lo_ = (p >= 2) ? s_vl[pa] : 0.0;
        up_ = (p <= K - 1) ? s_wf[me] : 0.0;
        r0 = s_xl[pa]; r1 = s_xf[me];
    }
    // Per step a block hands its neighbours three products each: to the block d to its right {u e01, q0, l idet}, to the block
    // d to its left {l e10, q1, u idet} (e01 = beta idet, e10 = gamma idet): 6 stores and 6 loads per step, 32-bit indices.
    int buf = 0;
    double q0 = 0.0, q1 = 0.0;
    const int S6 = 6 * S;
    for (int dd = 1;; dd <<= 1) {
        const double idet = 1.0 / (1.0 - beta * gamma);
        q0 = (r0 - beta * r1) * idet;
        q1 = (r1 - gamma * r0) * idet;
        if (dd >= K) break;                                             // uniform over the CTA
        double* Bf = pc + buf * S6 + me;
        Bf[0] = up_ * beta * idet; Bf[S] = q0; Bf[2 * S] = lo_ * idet;
        Bf[3 * S] = lo_ * gamma * idet; Bf[4 * S] = q1; Bf[5 * S] = up_ * idet;
        // couplings below 1e-30 of the unit diagonal are invisible in fp64: once every block of the CTA's lines is decoupled
        // (decayed spikes) the remaining steps would change nothing
        if (!__syncthreads_or(fabs(lo_) > 1e-30 || fabs(up_) > 1e-30)) break;
        if (p >= 1) {
            double ln = 0.0, un = 0.0;
            const int off = dd * pst;
            if (p - dd >= 1) {
                const double* Lp = Bf - off;
                beta = fma(lo_, Lp[0], beta);
                r0 = fma(-lo_, Lp[S], r0);
                ln = -lo_ * Lp[2 * S];
            }
            if (p + dd <= K) {
                const double* Rp = Bf + off;
                gamma = fma(up_, Rp[3 * S], gamma);
                r1 = fma(-up_, Rp[4 * S], r1);
                un = -up_ * Rp[5 * S];
            }
            lo_ = ln; up_ = un;
        }
        buf ^= 1;
    }
    s_t[me] = q1;                                                       // t_p = x_first_p
    __syncthreads();
    const double yL = (p >= 1) ? q0 : 0.0;                              // s_p = x_last_{p-1}
    const double yR = (p <= P - 2) ? s_t[me + pst] : 0.0;               // t_{p+1} = x_first_{p+1}
#pragma unroll
    for (int jj = 0; jj < M; ++jj) D_[jj] = fma(-A_[jj], yR, fma(-F_[jj], yL, D_[jj]));   // Eq.(8): x = xt - v yL - w yR
    // Acceptance test.  The neighbours' ACTUAL end values (not the reduced system's idea of them) and the coefficients once
    // more (they were read a moment ago: L1 / L2): the componentwise backward error of the line's equations in this
    // thread's rows.  NaN fails every comparison.
    s_xf[me] = D_[0]; s_xl[me] = D_[M - 1];                             // s_xf / s_xl were last read before the first barrier of the PCR
    if (!tame && valid) s_bad[L + lt] = 1;                              // benign race: every writer stores 1
    __syncthreads();
    const double xprev = (p >= 1) ? s_xl[me - pst] : 0.0, xnext = (p <= P - 2) ? s_xf[me + pst] : 0.0;
    bool bad = false;
    const bool check = s_bad[L + lt] != 0;                              // a line of tame blocks only is accepted as it is: no second read
#pragma unroll
    for (int jj = 0; jj < M; ++jj) {
        if (check && valid && jj < m) {
            const long long e = e0 + (long long)jj * G.row_stride;
            const double av = __ldg(G.a + e), bv = __ldg(G.b + e), cv = __ldg(G.c + e), dv = __ldg(G.d + e);
            const double xlo = (jj == 0) ? xprev : D_[jj > 0 ? jj - 1 : 0];
            const double xhi = (jj + 1 < m) ? D_[jj + 1 < M ? jj + 1 : jj] : xnext;
            const double t1 = (jj == 0 && p == 0) ? 0.0 : av * xlo, t2 = bv * D_[jj], t3 = (jj == m - 1 && p == P - 1) ? 0.0 : cv * xhi;
            const double res = (t1 + t2) + (t3 - dv);
            if (!(fabs(res) <= kGeneralBackwardError * (fabs(t1) + fabs(t2) + fabs(t3) + fabs(dv)))) bad = true;
        }
    }
    if (bad) s_bad[lt] = 1;
    __syncthreads();
    if (s_bad[lt] != 0) {
        if (p == 0 && valid) {
            const unsigned slot = atomicAdd(G.fb_count, 1u);
            if (slot < G.fb_cap) G.fb_lines[slot] = (unsigned)((long long)o * G.W + l);
            G.fb_flag[(long long)o * G.W + l] = 1;
        }
        return;                                                         // nothing of this line is written: k_general_lines solves it
    }
#pragma unroll
    for (int jj = 0; jj < M; ++jj)
        if (valid && jj < m) G.d[e0 + (long long)jj * G.row_stride] = D_[jj];
}

// One thread per line, diagonal pivoting over the WHOLE line, two passes (forward: modified diagonal, modified right-hand
// side and pivot types to the workspace; backward: substitution) -- the robust path:
//   LIST = true : the lines the partition kernel gave up on (G.fb_lines[0 .. *G.fb_count));
//   LIST = false: every line (the pivoting baseline, TDX_GENERAL_TWO_PASS=1, and lines too short or too long to partition);
//   CYC         : periodic lines -- a of the first row couples to the last row, c of the last row to the first: rank-1
//                 split of Eq.(3), A = A' + u v^T with u = (gamma, 0, .., 0, c_{n-1}), v = (1, 0, .., 0, a_0 / gamma);
//                 A' y = d and A' q = u by the same elimination, x = y - q (v.y) / (1 + v.q).  For matrices that are not
//                 dominant the split is only as good as A' is conditioned, which depends on gamma: the result is checked
//                 for cancellation (max |q s| against max |x|) BEFORE it is written and the line is redone with another
//                 gamma (sign flipped, doubled) when it lost more than three digits that way; d stays intact until then.
// Workspace, indexed like the field: bm (modified diagonal, doubles), fg (pivot type, bytes); CYC: qv (q) and dv (y).
// Pivot types: 0 = 1x1 pivot row, 1 = first row of a 2x2 pivot, 2 = second row.  Criterion: see the head of this file.
template <bool PIVOT, bool LIST, bool CYC>
__global__ void __launch_bounds__(128) k_general_lines(GeneralArgs G, double* __restrict__ bm, unsigned char* __restrict__ fg, double* __restrict__ qv,
                                                       double* __restrict__ dv) {
    if (general_deselected(G)) return;
    const double kappa = 0.6180339887498949;
    const int n = G.n;
    const long long rs = G.row_stride;
    // LIST: few listed lines are taken from the list (their threads read lines far apart: about three times the cost per line
    // of neighbouring lines); when more than a third of all lines are listed, every line is visited in memory order instead
    // and the accepted ones skipped (one flag byte per line), so the worst case costs what the kernel costs over all lines.
    const long long listed = LIST ? (long long)min(*G.fb_count, G.fb_cap) : 0;
    const bool dense = LIST && listed * 3 > (long long)G.fb_cap;
    const long long cnt = LIST ? (dense ? (long long)G.fb_cap : listed) : G.W;
    double* const rhs = CYC ? dv : G.d;                                 // where the modified right-hand side / y lives
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < cnt; s += (long long)gridDim.x * blockDim.x) {
        long long o, l;
        if (LIST) {
            const unsigned id = dense ? (unsigned)s : G.fb_lines[s];
            if (dense && G.fb_flag[id] == 0) continue;
            o = id / G.W; l = id - o * G.W;
        }
        else { o = blockIdx.y; l = s; }
        const long long base = o * G.outer_stride + l * G.lane_stride;
        const long long qe = base + (long long)(n - 1) * rs;              // last row
        double gamma = 0.0, g = 0.0, cn = 0.0, a0 = 0.0;
        if (CYC) {
            a0 = G.a[base]; cn = G.c[qe];
            const double sc = fabs(G.b[base]) + fabs(a0) + fabs(cn);
            gamma = (G.b[base] >= 0.0 ? -1.0 : 1.0) * (sc > 0.0 ? sc : 1.0);
        }
      for (int attempt = 0; attempt < (CYC ? 4 : 1); ++attempt) {
        if (CYC) g = a0 / gamma;
        auto bval = [&](long long q, int j) -> double {                   // diagonal of A' (CYC: corner rows shifted)
            double v = G.b[q];
            if (CYC && j == 0) v -= gamma;
            if (CYC && j == n - 1) v -= cn * g;
            return v;
        };
        double b0 = bval(base, 0), c0 = (n > 1) ? G.c[base] : 0.0, d0 = G.d[base], u0 = CYC ? gamma : 0.0;
        double a1 = 0.0, b1 = 1.0, c1 = 0.0, d1 = 0.0, u1 = 0.0, a2 = 0.0, b2 = 1.0, c2 = 0.0, d2 = 0.0, u2 = 0.0;
        if (n > 1) { const long long q = base + rs; a1 = G.a[q]; b1 = bval(q, 1); c1 = (n > 2) ? G.c[q] : 0.0; d1 = G.d[q]; u1 = (CYC && n == 2) ? cn : 0.0; }
        if (n > 2) { const long long q = base + 2 * rs; a2 = G.a[q]; b2 = bval(q, 2); c2 = (n > 3) ? G.c[q] : 0.0; d2 = G.d[q]; u2 = (CYC && n == 3) ? cn : 0.0; }
        bool second = false;
        for (int j = 0; j < n; ++j) {
            unsigned char f = 0;
            if (second) { f = 2; second = false; }
            else {
                bool one = true;
                if (PIVOT) {
                    const double sigma = fmax(fmax(fabs(c0), fabs(a1)), fmax(fabs(b1), fmax(fabs(c1), fabs(a2))));
                    one = fabs(b0) * sigma >= kappa * fabs(c0 * a1);
                }
                if (one) {
                    const double mlt = a1 / b0;
                    b1 = fma(-mlt, c0, b1); d1 = fma(-mlt, d0, d1);
                    if (CYC) u1 = fma(-mlt, u0, u1);
                } else {
                    f = 1; second = true;
                    const double t = a2 / (b0 * b1 - a1 * c0);
                    b2 = fma(-t, b0 * c1, b2);
                    d2 = fma(-t, b0 * d1 - a1 * d0, d2);
                    if (CYC) u2 = fma(-t, b0 * u1 - a1 * u0, u2);
                }
            }
            const long long q = base + (long long)j * rs;
            bm[q] = b0; rhs[q] = d0; fg[q] = f;
            if (CYC) qv[q] = u0;
            b0 = b1; c0 = c1; d0 = d1; u0 = u1;
            a1 = a2; b1 = b2; c1 = c2; d1 = d2; u1 = u2;
            if (j + 3 < n) {
                const long long q3 = base + (long long)(j + 3) * rs;
                a2 = G.a[q3]; b2 = bval(q3, j + 3); c2 = (j + 4 < n) ? G.c[q3] : 0.0; d2 = G.d[q3]; u2 = (CYC && j + 3 == n - 1) ? cn : 0.0;
            } else { a2 = 0.0; b2 = 1.0; c2 = 0.0; d2 = 0.0; u2 = 0.0; }
        }
        double xn = 0.0, pend = 0.0, zn = 0.0, zpend = 0.0, ylast = 0.0, qlast = 0.0;
        for (int j = n - 1; j >= 0; --j) {
            const long long q = base + (long long)j * rs;
            const unsigned char f = fg[q];
            double x, z = 0.0;
            if (f == 0) {
                const double cj = (j < n - 1) ? G.c[q] : 0.0, ib = 1.0 / bm[q];
                x = (rhs[q] - cj * xn) * ib;
                if (CYC) z = (qv[q] - cj * zn) * ib;
            } else if (f == 2) {                                        // rows j-1, j: [[b0, c0],[a1, b1]] (x_{j-1}, x_j) = (d_{j-1}, d_j - c_j x_{j+1})
                const long long pq = q - rs;
                const double pb0 = bm[pq], pc0 = G.c[pq], pa1 = G.a[q], pb1 = bm[q];
                const double cj = (j < n - 1) ? G.c[q] : 0.0;
                const double idet = 1.0 / (pb0 * pb1 - pa1 * pc0);
                const double r1 = rhs[pq], r2 = rhs[q] - cj * xn;
                x = (pb0 * r2 - pa1 * r1) * idet;
                pend = (pb1 * r1 - pc0 * r2) * idet;
                if (CYC) {
                    const double s1 = qv[pq], s2 = qv[q] - cj * zn;
                    z = (pb0 * s2 - pa1 * s1) * idet;
                    zpend = (pb1 * s1 - pc0 * s2) * idet;
                }
            } else { x = pend; z = zpend; }
            rhs[q] = x;
            if (CYC) { qv[q] = z; if (j == n - 1) { ylast = x; qlast = z; } }
            xn = x; zn = z;
        }
        if (CYC) {                                                      // xn = y_0, zn = q_0
            const double sfac = (xn + g * ylast) / (1.0 + zn + g * qlast);
            double mx = 0.0, mq = 0.0;
            for (int j = 0; j < n; ++j) { const long long q = base + (long long)j * rs; const double t = qv[q] * sfac; mq = fmax(mq, fabs(t)); mx = fmax(mx, fabs(rhs[q] - t)); }
            const bool ok = (mq <= 1e3 * mx) || (mq == 0.0);            // NaN fails: retried, written as it is on the last attempt
            if (ok || attempt == 3) {
                for (int j = 0; j < n; ++j) { const long long q = base + (long long)j * rs; G.d[q] = fma(-qv[q], sfac, rhs[q]); }
                break;
            }
            gamma *= -2.0;
        }
      }
    }
}

}  // namespace tdx
