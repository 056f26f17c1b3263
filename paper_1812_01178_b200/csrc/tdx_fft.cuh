// tdx_fft.cuh -- the transforms around the Poisson y-solves ("half-range cosine transform in the
// streamwise x-direction and Fourier transform in the spanwise z-direction ... after which the pseudo-pressure is
// obtained via inverse transforms"; L172: their modified wavenumbers shift the y-systems).  SURVEY 8(f) N2.
//
// Both transforms are HBM-bound passes over the field (8 B read + 8 B written per real value), in fp64, with no
// transpose: the z transform works on lines whose stride is nx*ny, the x transform on unit-stride lines.
//
//   core        radix-8/4/2 Stockham FFT of N = 2^k complex points held 8 per thread in registers (thread t of the
//               N/8 threads of a transform holds points t + kk*N/8); between passes the points are exchanged through
//               shared memory (one write + one read of 16 B per point per pass).  Twiddles: one table load
//               (W_N^q, plan-time sincospi) per butterfly, powers by multiplication.
//   k_rfft_z    two adjacent x-values (one 16-byte load) are the re/im parts of ONE complex transform along z
//               ("two real transforms for one complex"); the spectra of the two real columns are separated at the
//               end, A_m = (Z_m + conj Z_{N-m})/2, B_m = (Z_m - conj Z_{N-m})/(2i), and stored as complex128
//               [nm][ny][nx].  CTA = C column pairs (C*32 contiguous bytes of every z-row) x N/8 threads.
//   k_irfft_z   the reverse: Z_m = A_m + i B_m, Z_{N-m} = conj A_m + i conj B_m, inverse transform by the
//               swap-re/im identity, 1/N scaling, 16-byte stores of the two real columns.
//   k_dct_x     cosine transform (DCT-II, reading T1 of DESIGN.md) of two adjacent x-lines at once through one
//               N-point complex FFT (Makhoul's even/odd permutation v_n = x_{2n}, v_{N-1-n} = x_{2n+1}; then
//               X_k = Re(w_k V_k), X_{N-k} = -Im(w_k V_k), w_k = exp(-i pi k / 2N)).  The CTA's lines are one
//               contiguous piece of HBM: they come in and go out as 1-D bulk copies (cp.async.bulk, TMA engine).
//               Inverse (DCT-III scaled so that it inverts the forward one): V_k = conj(w_k)(X_k - i X_{N-k}).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "tdx_tma.cuh"

namespace tdx {

// ---- complex helpers --------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmul_mi(double2 a) { return make_double2(a.y, -a.x); }      // a * (-i)

// forward DFTs (exp(-2 pi i ...)), natural order in and out
__device__ __forceinline__ void dft2(double2& a, double2& b) { const double2 t = csub(a, b); a = cadd(a, b); b = t; }
__device__ __forceinline__ void dft4(double2& a0, double2& a1, double2& a2, double2& a3) {
    const double2 s0 = cadd(a0, a2), d0 = csub(a0, a2), s1 = cadd(a1, a3), d1 = cmul_mi(csub(a1, a3));
    a0 = cadd(s0, s1); a2 = csub(s0, s1); a1 = cadd(d0, d1); a3 = csub(d0, d1);
}
__device__ __forceinline__ void dft8(double2 (&v)[8]) {
    const double h = 0.70710678118654752440;
    double2 b0 = cadd(v[0], v[4]), b4 = csub(v[0], v[4]);
    double2 b1 = cadd(v[1], v[5]), b5 = csub(v[1], v[5]);
    double2 b2 = cadd(v[2], v[6]), b6 = csub(v[2], v[6]);
    double2 b3 = cadd(v[3], v[7]), b7 = csub(v[3], v[7]);
    b5 = make_double2((b5.x + b5.y) * h, (b5.y - b5.x) * h);          // * W8^1 = (1 - i)/sqrt2
    b6 = cmul_mi(b6);                                                 // * W8^2 = -i
    b7 = make_double2((b7.y - b7.x) * h, -(b7.x + b7.y) * h);         // * W8^3 = (-1 - i)/sqrt2
    dft4(b0, b1, b2, b3);                                             // even outputs X0 X2 X4 X6
    dft4(b4, b5, b6, b7);                                             // odd outputs  X1 X3 X5 X7
    v[0] = b0; v[2] = b1; v[4] = b2; v[6] = b3;
    v[1] = b4; v[3] = b5; v[5] = b6; v[7] = b7;
}

// 16-point DFT as 4 x 4 (Cooley-Tukey): inner DFT4 over n1 of x[4 n1 + q], twiddle W16^(q k1), outer DFT4 over q.
__device__ __forceinline__ void dft16(double2 (&v)[16]) {
    const double h = 0.70710678118654752440, c1 = 0.92387953251128675613, s1 = 0.38268343236508977173;
#pragma unroll
    for (int q = 0; q < 4; ++q) dft4(v[q], v[q + 4], v[q + 8], v[q + 12]);          // v[q + 4 k1] = inner output k1 of column q
    // twiddles W16^(q k1), q, k1 in 1..3
    v[1 + 4] = cmul(v[1 + 4], make_double2(c1, -s1));                                // W^1
    v[1 + 8] = make_double2((v[1 + 8].x + v[1 + 8].y) * h, (v[1 + 8].y - v[1 + 8].x) * h);   // W^2
    v[1 + 12] = cmul(v[1 + 12], make_double2(s1, -c1));                              // W^3
    v[2 + 4] = make_double2((v[2 + 4].x + v[2 + 4].y) * h, (v[2 + 4].y - v[2 + 4].x) * h);   // W^2
    v[2 + 8] = cmul_mi(v[2 + 8]);                                                    // W^4 = -i
    v[2 + 12] = make_double2((v[2 + 12].y - v[2 + 12].x) * h, -(v[2 + 12].x + v[2 + 12].y) * h);   // W^6
    v[3 + 4] = cmul(v[3 + 4], make_double2(s1, -c1));                                // W^3
    v[3 + 8] = make_double2((v[3 + 8].y - v[3 + 8].x) * h, -(v[3 + 8].x + v[3 + 8].y) * h);   // W^6
    v[3 + 12] = cmul(v[3 + 12], make_double2(-c1, s1));                              // W^9
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);   // slot 4 k1 + k2 = X[k1 + 4 k2]
    // to natural order: X[k] sits in slot 4 (k & 3) + (k >> 2)
    double2 o[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) o[k] = v[4 * (k & 3) + (k >> 2)];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = o[k];
}

// One Stockham pass of radix R on the K register points of thread t (slot kk = point t + kk*N/K).  NS = product of
// the radices of the earlier passes.  Butterfly s (of B = K/R) takes slots s + r*B, r < R; its index is j = t + s*N/K.
// pos[kk] receives the position the slot's value has after the pass: (j - j%NS)*R + j%NS + r*NS.
template <int N, int K, int R, int NS, int TWS = 1>
__device__ __forceinline__ void fft_pass(double2 (&v)[K], int (&pos)[K], int t, const double2* __restrict__ tw) {
    constexpr int T = N / K, B = K / R;
#pragma unroll
    for (int s = 0; s < B; ++s) {
        const int j = t + s * T;
        const int jm = j & (NS - 1);
        double2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = v[s + r * B];
        if (NS > 1) {
            const double2 w1 = __ldg(tw + TWS * (jm * (N / (NS * R))));      // TWS: stride into a table of TWS*N roots
            x[1] = cmul(x[1], w1);
            if constexpr (R >= 4) {
                const double2 w2 = cmul(w1, w1), w3 = cmul(w2, w1);
                x[2] = cmul(x[2], w2); x[3] = cmul(x[3], w3);
                if constexpr (R >= 8) {
                    const double2 w4 = cmul(w2, w2), w5 = cmul(w4, w1), w6 = cmul(w4, w2), w7 = cmul(w4, w3);
                    x[4] = cmul(x[4], w4); x[5] = cmul(x[5], w5); x[6] = cmul(x[6], w6); x[7] = cmul(x[7], w7);
                    if constexpr (R >= 16) {
                        const double2 w8 = cmul(w4, w4);
                        x[8] = cmul(x[8], w8); x[9] = cmul(x[9], cmul(w8, w1)); x[10] = cmul(x[10], cmul(w8, w2));
                        x[11] = cmul(x[11], cmul(w8, w3)); x[12] = cmul(x[12], cmul(w8, w4)); x[13] = cmul(x[13], cmul(w8, w5));
                        x[14] = cmul(x[14], cmul(w8, w6)); x[15] = cmul(x[15], cmul(w8, w7));
                    }
                }
            }
        }
        if constexpr (R == 2) dft2(x[0], x[1]);
        else if constexpr (R == 4) dft4(x[0], x[1], x[2], x[3]);
        else if constexpr (R == 8) dft8(x);
        else dft16(x);
        const int base = (j - jm) * R + jm;
#pragma unroll
        for (int r = 0; r < R; ++r) { v[s + r * B] = x[r]; pos[s + r * B] = base + r * NS; }
    }
}

// Whole transform: passes of radix K while they fit, then the remaining factor.  SM maps a position to a shared-memory
// slot (SM::at(pos)).  On return v[kk] = X[t + kk*N/K] (the last pass leaves its outputs in the slots they came from).
// Every pass but the last ends with: scatter to shared, barrier, gather, barrier.
template <int N, int K, int NS, class SM>
__device__ __forceinline__ void fft_regs(double2 (&v)[K], int t, const double2* __restrict__ tw, const SM& sm) {
    constexpr int T = N / K;
    constexpr int R = (N / NS >= K) ? K : (N / NS);
    int pos[K];
    fft_pass<N, K, R, NS>(v, pos, t, tw);
    if constexpr (NS * R < N) {
#pragma unroll
        for (int kk = 0; kk < K; ++kk) *sm.at(pos[kk]) = v[kk];
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < K; ++kk) v[kk] = *sm.at(t + kk * T);
        __syncthreads();
        fft_regs<N, K, NS * R, SM>(v, t, tw, sm);
    }
}

// Three transforms of length M side by side in one thread (the sub-sequences x_{3m+r}, r = 0, 1, 2, of a transform of
// length N = 3M): the same passes in lockstep, sharing the barriers.  tw is the table of N-th roots (stride 3 gives the
// M-th roots).  sm[r] maps positions of sub-transform r.
template <int M, int K, int NS, class SM>
__device__ __forceinline__ void fft_regs3(double2 (&v)[3][K], int t, const double2* __restrict__ tw, const SM (&sm)[3]) {
    constexpr int T = M / K;
    constexpr int R = (M / NS >= K) ? K : (M / NS);
    int pos[K];
#pragma unroll
    for (int r = 0; r < 3; ++r) fft_pass<M, K, R, NS, 3>(v[r], pos, t, tw);
    if constexpr (NS * R < M) {
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int kk = 0; kk < K; ++kk) *sm[r].at(pos[kk]) = v[r][kk];
        __syncthreads();
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int kk = 0; kk < K; ++kk) v[r][kk] = *sm[r].at(t + kk * T);
        __syncthreads();
        fft_regs3<M, K, NS * R, SM>(v, t, tw, sm);
    }
}

// Radix-3 recombination X[k + s M] = sum_r W_3^{r s} W_N^{r k} F_r[k] (decimation in time by 3); in place: f_r -> X_s.
__device__ __forceinline__ void combine3(double2& f0, double2& f1, double2& f2, double2 w1, double2 w2) {
    const double hs = 0.86602540378443864676;                   // sqrt(3)/2
    const double2 b = cmul(f1, w1), c = cmul(f2, w2);
    const double2 s = cadd(b, c), d = csub(b, c);
    const double2 m = make_double2(f0.x - 0.5 * s.x, f0.y - 0.5 * s.y);
    const double2 rot = make_double2(hs * d.y, -hs * d.x);       // -i sqrt(3)/2 (b - c)
    f0 = cadd(f0, s);
    f1 = cadd(m, rot);                                           // a + w b + w^2 c, w = exp(-2 pi i / 3)
    f2 = csub(m, rot);
}

// shared-memory maps
struct SmCols {      // z transforms: [pos][C columns], column fastest
    double2* base; int C;
    __device__ __forceinline__ double2* at(int pos) const { return base + pos * C; }
};
template <int K>
struct SmPad {       // x transforms: one line pair, one pad slot per K (the first pass writes with stride K)
    double2* base;
    __device__ __forceinline__ double2* at(int pos) const { return base + pos + (pos >> (K == 16 ? 4 : 3)); }
};

// ---- plan-time tables ---------------------------------------------------------------------------------------------
// tw[q] = exp(-2 pi i q / N), q < N;  w4[k] = exp(-i pi k / (2N)), k <= N/2
__global__ void k_fft_tables(double2* __restrict__ tw, double2* __restrict__ w4, int N) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < N) { double s, c; sincospi(2.0 * (double)q / (double)N, &s, &c); tw[q] = make_double2(c, -s); }
    if (w4 && q <= N / 2) { double s, c; sincospi((double)q / (2.0 * (double)N), &s, &c); w4[q] = make_double2(c, -s); }
}

// ---- Fourier transform along z --------------------------------------------------------------------------------------
// in: real [nz=N][ny][nx]; out: complex128 [N/2+1][ny][nx].  grid (ceil(nx / 2C), ny), block (C, N/8).  nx even.
template <int N, int C, int K>
__global__ void __launch_bounds__(C * N / K) k_rfft_z(const double* __restrict__ in, double2* __restrict__ out, int nx, int ny,
                                                       const double2* __restrict__ tw, int pf) {
    constexpr int T = N / K, H = K / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* smb = reinterpret_cast<double2*>(smem_raw);
    const int c = threadIdx.x, t = threadIdx.y;
    const int j = blockIdx.y;
    const long long i0 = (long long)blockIdx.x * 2 * C + 2 * c;
    const bool act = i0 < nx;
    const size_t plane = (size_t)nx * ny;
    const double* src = in + (size_t)j * nx + i0;
    double2 v[K];
#pragma unroll
    for (int kk = 0; kk < K; ++kk)
        v[kk] = act ? __ldcs(reinterpret_cast<const double2*>(src + (size_t)(t + kk * T) * plane)) : make_double2(0.0, 0.0);
    if (pf > 0 && (c & 7) == 0) {                  // L2 prefetch of the tile the CTA `pf` launches ahead will load (one lane per 128 B)
        const long long lin = (long long)blockIdx.y * gridDim.x + blockIdx.x + pf;
        const long long by = lin / gridDim.x, bx = lin - by * gridDim.x;
        const long long pi = bx * 2 * C + 2 * c;
        if (by < ny && pi < nx) {
            const double* pb = in + (size_t)by * nx + pi;
#pragma unroll
            for (int kk = 0; kk < K; ++kk) asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + (size_t)(t + kk * T) * plane));
        }
    }
    const SmCols sm{smb + c, C};
    fft_regs<N, K, 1, SmCols>(v, t, tw, sm);
#pragma unroll
    for (int kk = 0; kk < K; ++kk) *sm.at(t + kk * T) = v[kk];
    __syncthreads();
    double2* dst = out + (size_t)j * nx + i0;
#pragma unroll
    for (int kk = 0; kk < H; ++kk) {
        const int m = t + kk * T;
        const double2 zm = *sm.at(m), zn = *sm.at((N - m) & (N - 1));
        if (act) {
            double2* o = dst + (size_t)m * plane;
            __stcs(o, make_double2(0.5 * (zm.x + zn.x), 0.5 * (zm.y - zn.y)));
            __stcs(o + 1, make_double2(0.5 * (zm.y + zn.y), 0.5 * (zn.x - zm.x)));
        }
    }
    if (t == 0 && act) {
        const double2 z = *sm.at(N / 2);
        double2* o = dst + (size_t)(N / 2) * plane;
        __stcs(o, make_double2(z.x, 0.0));
        __stcs(o + 1, make_double2(z.y, 0.0));
    }
}

// in: complex128 [N/2+1][ny][nx]; out: real [N][ny][nx] (includes the 1/N).  Same launch shape as k_rfft_z.
template <int N, int C, int K>
__global__ void __launch_bounds__(C * N / K) k_irfft_z(const double2* __restrict__ in, double* __restrict__ out, int nx, int ny,
                                                        const double2* __restrict__ tw, int pf) {
    constexpr int T = N / K, H = K / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* smb = reinterpret_cast<double2*>(smem_raw);
    const int c = threadIdx.x, t = threadIdx.y;
    const int j = blockIdx.y;
    const long long i0 = (long long)blockIdx.x * 2 * C + 2 * c;
    const bool act = i0 < nx;
    const size_t plane = (size_t)nx * ny;
    const double2* src = in + (size_t)j * nx + i0;
    const SmCols sm{smb + c, C};
    double2 a[H + 1], b[H + 1];
#pragma unroll
    for (int kk = 0; kk < H; ++kk) {
        const double2* p = src + (size_t)(t + kk * T) * plane;
        a[kk] = act ? __ldcs(p) : make_double2(0.0, 0.0);
        b[kk] = act ? __ldcs(p + 1) : make_double2(0.0, 0.0);
    }
    if (t == 0) {
        const double2* p = src + (size_t)(N / 2) * plane;
        a[H] = act ? __ldcs(p) : make_double2(0.0, 0.0);
        b[H] = act ? __ldcs(p + 1) : make_double2(0.0, 0.0);
    }
    if (pf > 0 && (c & 3) == 0) {                  // spectrum rows are 32 B per column pair: one lane per 128 B
        const long long lin = (long long)blockIdx.y * gridDim.x + blockIdx.x + pf;
        const long long by = lin / gridDim.x, bx = lin - by * gridDim.x;
        const long long pi = bx * 2 * C + 2 * c;
        if (by < ny && pi < nx) {
            const double2* pb = in + (size_t)by * nx + pi;
#pragma unroll
            for (int kk = 0; kk < H; ++kk) asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + (size_t)(t + kk * T) * plane));
            if (t == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + (size_t)(N / 2) * plane));
        }
    }
    // Z_m = A + iB, Z_{N-m} = conj A + i conj B; stored with re/im swapped (inverse transform by the swap identity)
#pragma unroll
    for (int kk = 0; kk < H; ++kk) {
        const int m = t + kk * T;
        if (m == 0) {
            *sm.at(0) = make_double2(b[kk].x, a[kk].x);
        } else {
            *sm.at(m) = make_double2(a[kk].y + b[kk].x, a[kk].x - b[kk].y);
            *sm.at(N - m) = make_double2(b[kk].x - a[kk].y, a[kk].x + b[kk].y);
        }
    }
    if (t == 0) *sm.at(N / 2) = make_double2(b[H].x, a[H].x);
    __syncthreads();
    double2 v[K];
#pragma unroll
    for (int kk = 0; kk < K; ++kk) v[kk] = *sm.at(t + kk * T);
    __syncthreads();
    fft_regs<N, K, 1, SmCols>(v, t, tw, sm);
    const double sc = 1.0 / (double)N;
    double* dst = out + (size_t)j * nx + i0;
    if (act) {
#pragma unroll
        for (int kk = 0; kk < K; ++kk)
            __stcs(reinterpret_cast<double2*>(dst + (size_t)(t + kk * T) * plane), make_double2(v[kk].y * sc, v[kk].x * sc));
    }
}

// ---- cosine transform along x -----------------------------------------------------------------------------------------
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(src)), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store_1d(void* dst, const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(reinterpret_cast<uint64_t>(dst)), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_1d(const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(reinterpret_cast<uint64_t>(src)), "r"(bytes) : "memory");
}

// field: [lines][N] doubles, in place.  CTA = LP line pairs (2*LP*N contiguous doubles) x N/8 threads per pair.
// Shared memory: LP * (N + N/8) double2 (the raw lines occupy the first LP*2N doubles of it) + one mbarrier.
template <int N, int LP, int INV, int K>
__global__ void __launch_bounds__(LP * N / K) k_dct_x(double* __restrict__ field, long long lines,
                                                       const double2* __restrict__ tw, const double2* __restrict__ w4, int pf) {
    constexpr int T = N / K, H = K / 2;
    constexpr int PSTR = N + N / K;                           // double2 slots per pair in the exchange layout
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* smb = reinterpret_cast<double2*>(smem_raw);
    double* raw = reinterpret_cast<double*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)LP * PSTR * 16);
    const int tid = threadIdx.x;
    const int p = tid / T, t = tid - p * T;
    const long long line0 = (long long)blockIdx.x * 2 * LP;
    const long long nl = min((long long)2 * LP, lines - line0);              // lines of this CTA (> 0)
    const uint32_t bytes = (uint32_t)(nl * N * 8);
    double* gsrc = field + (size_t)line0 * N;
    if (tid == 0) { mbar_init(bar, 1); mbar_fence_init(); }
    __syncthreads();
    if (tid == 0) {
        mbar_arrive_expect_tx(bar, bytes);
        bulk_load_1d(raw, gsrc, bytes, bar);
        if (pf > 0) {
            const long long l2 = line0 + (long long)pf * 2 * LP;
            if (l2 < lines) bulk_prefetch_1d(field + (size_t)l2 * N, (uint32_t)(min((long long)2 * LP, lines - l2) * N * 8));
        }
    }
    mbar_wait(bar, 0);
    const bool has_a = 2 * p < nl, has_b = 2 * p + 1 < nl;
    const double* la = raw + (size_t)p * 2 * N;
    const double* lb = la + N;
    const SmPad<K> sm{smb + (size_t)p * PSTR};
    double2 v[K];
    if (!INV) {
#pragma unroll
        for (int kk = 0; kk < K; ++kk) {
            const int n = t + kk * T;
            const int idx = (n < N / 2) ? 2 * n : 2 * (N - 1 - n) + 1;
            v[kk] = make_double2(has_a ? la[idx] : 0.0, has_b ? lb[idx] : 0.0);
        }
        __syncthreads();                                                       // raw lines consumed; the buffer becomes the exchange area
        fft_regs<N, K, 1, SmPad<K>>(v, t, tw, sm);
#pragma unroll
        for (int kk = 0; kk < K; ++kk) *sm.at(t + kk * T) = v[kk];
        __syncthreads();
        double2 zk[H + 1], zn[H + 1];
#pragma unroll
        for (int kk = 0; kk < H; ++kk) { const int k = t + kk * T; zk[kk] = *sm.at(k); zn[kk] = *sm.at((N - k) & (N - 1)); }
        if (t == 0) { zk[H] = *sm.at(N / 2); zn[H] = zk[H]; }
        __syncthreads();                                                       // spectrum consumed; the buffer becomes the raw lines again
        double* oa = raw + (size_t)p * 2 * N;
        double* ob = oa + N;
#pragma unroll
        for (int kk = 0; kk <= H; ++kk) {
            if (kk == H && t != 0) break;
            const int k = (kk == H) ? N / 2 : t + kk * T;
            // V_a = (Z_k + conj Z_{N-k})/2, V_b = (Z_k - conj Z_{N-k})/(2i)
            const double2 va = make_double2(0.5 * (zk[kk].x + zn[kk].x), 0.5 * (zk[kk].y - zn[kk].y));
            const double2 vb = make_double2(0.5 * (zk[kk].y + zn[kk].y), 0.5 * (zn[kk].x - zk[kk].x));
            const double2 w = __ldg(w4 + k);
            const double2 ya = cmul(w, va), yb = cmul(w, vb);
            oa[k] = ya.x; ob[k] = yb.x;                                        // X_k = Re(w_k V_k)
            if (k != 0 && k != N / 2) { oa[N - k] = -ya.y; ob[N - k] = -yb.y; }   // X_{N-k} = -Im(w_k V_k)
        }
    } else {
        double xa[H + 1], xan[H + 1], xb[H + 1], xbn[H + 1];
#pragma unroll
        for (int kk = 0; kk <= H; ++kk) {
            if (kk == H && t != 0) break;
            const int k = (kk == H) ? N / 2 : t + kk * T;
            xa[kk] = has_a ? la[k] : 0.0; xb[kk] = has_b ? lb[k] : 0.0;
            xan[kk] = (k == 0 || !has_a) ? 0.0 : la[N - k];
            xbn[kk] = (k == 0 || !has_b) ? 0.0 : lb[N - k];
        }
        __syncthreads();
        // V_k = conj(w_k)(X_k - i X_{N-k}); Z_k = Va_k + i Vb_k; Z_{N-k} = conj(Va_k) + i conj(Vb_k); stored swapped
#pragma unroll
        for (int kk = 0; kk <= H; ++kk) {
            if (kk == H && t != 0) break;
            const int k = (kk == H) ? N / 2 : t + kk * T;
            const double2 w = __ldg(w4 + k);
            const double2 wc = make_double2(w.x, -w.y);
            const double2 va = cmul(wc, make_double2(xa[kk], -xan[kk]));
            const double2 vb = cmul(wc, make_double2(xb[kk], -xbn[kk]));
            *sm.at(k) = make_double2(va.y + vb.x, va.x - vb.y);
            if (k != 0 && k != N / 2) *sm.at(N - k) = make_double2(vb.x - va.y, va.x + vb.y);
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < K; ++kk) v[kk] = *sm.at(t + kk * T);
        __syncthreads();
        fft_regs<N, K, 1, SmPad<K>>(v, t, tw, sm);
        __syncthreads();                                                       // (fft_regs ends on a gather barrier only if it had > 1 pass)
        const double sc = 1.0 / (double)N;
        double* oa = raw + (size_t)p * 2 * N;
        double* ob = oa + N;
#pragma unroll
        for (int kk = 0; kk < K; ++kk) {
            const int n = t + kk * T;
            const int idx = (n < N / 2) ? 2 * n : 2 * (N - 1 - n) + 1;
            oa[idx] = v[kk].y * sc; ob[idx] = v[kk].x * sc;                    // un-swap: re of the inverse is the stored im
        }
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
        bulk_store_1d(gsrc, raw, bytes);
        tma_commit();
        tma_wait_read<0>();
    }
}

// ---- lengths N = 3 * 2^k (the paper's own grid is 3072 x 256 x 768) ------------------------------
// Decimation in time by 3: every thread runs the three M-point sub-transforms of its points side by side (8 points each)
// and recombines them in registers (combine3); loads, stores and the pairing of the two real transforms are as above.
template <int N, int C>
__global__ void __launch_bounds__(C * N / 24, (C * N / 24 <= 256) ? 2 : 1) k_rfft_z3(const double* __restrict__ in, double2* __restrict__ out, int nx, int ny,
                                                         const double2* __restrict__ tw) {
    constexpr int K = 8, M = N / 3, T = M / K;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* smb = reinterpret_cast<double2*>(smem_raw);
    const int c = threadIdx.x, t = threadIdx.y, j = blockIdx.y;
    const long long i0 = (long long)blockIdx.x * 2 * C + 2 * c;
    const bool act = i0 < nx;
    const size_t plane = (size_t)nx * ny;
    const double* src = in + (size_t)j * nx + i0;
    double2 v[3][K];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int kk = 0; kk < K; ++kk)
            v[r][kk] = act ? __ldcs(reinterpret_cast<const double2*>(src + (size_t)(3 * (t + kk * T) + r) * plane)) : make_double2(0.0, 0.0);
    const SmCols sm[3] = {{smb + c, C}, {smb + (size_t)M * C + c, C}, {smb + (size_t)2 * M * C + c, C}};
    fft_regs3<M, K, 1, SmCols>(v, t, tw, sm);
    const SmCols all{smb + c, C};
#pragma unroll
    for (int kk = 0; kk < K; ++kk) {
        const int k = t + kk * T;
        combine3(v[0][kk], v[1][kk], v[2][kk], __ldg(tw + k), __ldg(tw + 2 * k));
        *all.at(k) = v[0][kk]; *all.at(k + M) = v[1][kk]; *all.at(k + 2 * M) = v[2][kk];
    }
    __syncthreads();
    double2* dst = out + (size_t)j * nx + i0;
#pragma unroll
    for (int kk = 0; kk < 3 * K / 2; ++kk) {
        const int m = t + kk * T;
        const double2 zm = *all.at(m), zn = *all.at(m == 0 ? 0 : N - m);
        if (act) {
            double2* o = dst + (size_t)m * plane;
            __stcs(o, make_double2(0.5 * (zm.x + zn.x), 0.5 * (zm.y - zn.y)));
            __stcs(o + 1, make_double2(0.5 * (zm.y + zn.y), 0.5 * (zn.x - zm.x)));
        }
    }
    if (t == 0 && act) {
        const double2 z = *all.at(N / 2);
        double2* o = dst + (size_t)(N / 2) * plane;
        __stcs(o, make_double2(z.x, 0.0));
        __stcs(o + 1, make_double2(z.y, 0.0));
    }
}

template <int N, int C>
__global__ void __launch_bounds__(C * N / 24, (C * N / 24 <= 256) ? 2 : 1) k_irfft_z3(const double2* __restrict__ in, double* __restrict__ out, int nx, int ny,
                                                          const double2* __restrict__ tw) {
    constexpr int K = 8, M = N / 3, T = M / K;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* smb = reinterpret_cast<double2*>(smem_raw);
    const int c = threadIdx.x, t = threadIdx.y, j = blockIdx.y;
    const long long i0 = (long long)blockIdx.x * 2 * C + 2 * c;
    const bool act = i0 < nx;
    const size_t plane = (size_t)nx * ny;
    const double2* src = in + (size_t)j * nx + i0;
    const SmCols all{smb + c, C};
#pragma unroll
    for (int kk = 0; kk <= 3 * K / 2; ++kk) {
        if (kk == 3 * K / 2 && t != 0) break;
        const int m = (kk == 3 * K / 2) ? N / 2 : t + kk * T;
        const double2* p = src + (size_t)m * plane;
        const double2 a = act ? __ldcs(p) : make_double2(0.0, 0.0), b = act ? __ldcs(p + 1) : make_double2(0.0, 0.0);
        if (m == 0 || m == N / 2) {
            *all.at(m) = make_double2(b.x, a.x);
        } else {
            *all.at(m) = make_double2(a.y + b.x, a.x - b.y);
            *all.at(N - m) = make_double2(b.x - a.y, a.x + b.y);
        }
    }
    __syncthreads();
    double2 v[3][K];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int kk = 0; kk < K; ++kk) v[r][kk] = *all.at(3 * (t + kk * T) + r);
    __syncthreads();
    const SmCols sm[3] = {{smb + c, C}, {smb + (size_t)M * C + c, C}, {smb + (size_t)2 * M * C + c, C}};
    fft_regs3<M, K, 1, SmCols>(v, t, tw, sm);
    const double sc = 1.0 / (double)N;
    double* dst = out + (size_t)j * nx + i0;
#pragma unroll
    for (int kk = 0; kk < K; ++kk) {
        const int k = t + kk * T;
        combine3(v[0][kk], v[1][kk], v[2][kk], __ldg(tw + k), __ldg(tw + 2 * k));
        if (act) {
#pragma unroll
            for (int s = 0; s < 3; ++s)
                __stcs(reinterpret_cast<double2*>(dst + (size_t)(k + s * M) * plane), make_double2(v[s][kk].y * sc, v[s][kk].x * sc));
        }
    }
}

template <int N, int LP, int INV>
__global__ void __launch_bounds__(LP * N / 24) k_dct_x3(double* __restrict__ field, long long lines,
                                                         const double2* __restrict__ tw, const double2* __restrict__ w4, int pf) {
    constexpr int K = 8, M = N / 3, T = M / K, H3 = 3 * K / 2;
    constexpr int PSTR = N + N / 8;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* smb = reinterpret_cast<double2*>(smem_raw);
    double* raw = reinterpret_cast<double*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)LP * PSTR * 16);
    const int tid = threadIdx.x;
    const int p = tid / T, t = tid - p * T;
    const long long line0 = (long long)blockIdx.x * 2 * LP;
    const long long nl = min((long long)2 * LP, lines - line0);
    const uint32_t bytes = (uint32_t)(nl * N * 8);
    double* gsrc = field + (size_t)line0 * N;
    if (tid == 0) { mbar_init(bar, 1); mbar_fence_init(); }
    __syncthreads();
    if (tid == 0) {
        mbar_arrive_expect_tx(bar, bytes);
        bulk_load_1d(raw, gsrc, bytes, bar);
        if (pf > 0) {
            const long long l2 = line0 + (long long)pf * 2 * LP;
            if (l2 < lines) bulk_prefetch_1d(field + (size_t)l2 * N, (uint32_t)(min((long long)2 * LP, lines - l2) * N * 8));
        }
    }
    mbar_wait(bar, 0);
    const bool has_a = 2 * p < nl, has_b = 2 * p + 1 < nl;
    double* la = raw + (size_t)p * 2 * N;
    double* lb = la + N;
    const SmPad<8> all{smb + (size_t)p * PSTR};
    const SmPad<8> sm[3] = {{smb + (size_t)p * PSTR}, {smb + (size_t)p * PSTR + (M + M / 8)}, {smb + (size_t)p * PSTR + 2 * (M + M / 8)}};
    double2 v[3][K];
    if (!INV) {
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int kk = 0; kk < K; ++kk) {
                const int n = 3 * (t + kk * T) + r;
                const int idx = (n < N / 2) ? 2 * n : 2 * (N - 1 - n) + 1;
                v[r][kk] = make_double2(has_a ? la[idx] : 0.0, has_b ? lb[idx] : 0.0);
            }
        __syncthreads();
        fft_regs3<M, K, 1, SmPad<8>>(v, t, tw, sm);
#pragma unroll
        for (int kk = 0; kk < K; ++kk) {
            const int k = t + kk * T;
            combine3(v[0][kk], v[1][kk], v[2][kk], __ldg(tw + k), __ldg(tw + 2 * k));
            *all.at(k) = v[0][kk]; *all.at(k + M) = v[1][kk]; *all.at(k + 2 * M) = v[2][kk];
        }
        __syncthreads();
        double2 zk[H3 + 1], zn[H3 + 1];
#pragma unroll
        for (int kk = 0; kk < H3; ++kk) { const int k = t + kk * T; zk[kk] = *all.at(k); zn[kk] = *all.at(k == 0 ? 0 : N - k); }
        if (t == 0) { zk[H3] = *all.at(N / 2); zn[H3] = zk[H3]; }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk <= H3; ++kk) {
            if (kk == H3 && t != 0) break;
            const int k = (kk == H3) ? N / 2 : t + kk * T;
            const double2 va = make_double2(0.5 * (zk[kk].x + zn[kk].x), 0.5 * (zk[kk].y - zn[kk].y));
            const double2 vb = make_double2(0.5 * (zk[kk].y + zn[kk].y), 0.5 * (zn[kk].x - zk[kk].x));
            const double2 w = __ldg(w4 + k);
            const double2 ya = cmul(w, va), yb = cmul(w, vb);
            la[k] = ya.x; lb[k] = yb.x;
            if (k != 0 && k != N / 2) { la[N - k] = -ya.y; lb[N - k] = -yb.y; }
        }
    } else {
        double xa[H3 + 1], xan[H3 + 1], xb[H3 + 1], xbn[H3 + 1];
#pragma unroll
        for (int kk = 0; kk <= H3; ++kk) {
            if (kk == H3 && t != 0) break;
            const int k = (kk == H3) ? N / 2 : t + kk * T;
            xa[kk] = has_a ? la[k] : 0.0; xb[kk] = has_b ? lb[k] : 0.0;
            xan[kk] = (k == 0 || !has_a) ? 0.0 : la[N - k];
            xbn[kk] = (k == 0 || !has_b) ? 0.0 : lb[N - k];
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk <= H3; ++kk) {
            if (kk == H3 && t != 0) break;
            const int k = (kk == H3) ? N / 2 : t + kk * T;
            const double2 w = __ldg(w4 + k);
            const double2 wc = make_double2(w.x, -w.y);
            const double2 va = cmul(wc, make_double2(xa[kk], -xan[kk]));
            const double2 vb = cmul(wc, make_double2(xb[kk], -xbn[kk]));
            *all.at(k) = make_double2(va.y + vb.x, va.x - vb.y);
            if (k != 0 && k != N / 2) *all.at(N - k) = make_double2(vb.x - va.y, va.x + vb.y);
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int kk = 0; kk < K; ++kk) v[r][kk] = *all.at(3 * (t + kk * T) + r);
        __syncthreads();
        fft_regs3<M, K, 1, SmPad<8>>(v, t, tw, sm);
        __syncthreads();
        const double sc = 1.0 / (double)N;
#pragma unroll
        for (int kk = 0; kk < K; ++kk) {
            const int k = t + kk * T;
            combine3(v[0][kk], v[1][kk], v[2][kk], __ldg(tw + k), __ldg(tw + 2 * k));
#pragma unroll
            for (int s = 0; s < 3; ++s) {
                const int n = k + s * M;
                const int idx = (n < N / 2) ? 2 * n : 2 * (N - 1 - n) + 1;
                la[idx] = v[s][kk].y * sc; lb[idx] = v[s][kk].x * sc;
            }
        }
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
        bulk_store_1d(gsrc, raw, bytes);
        tma_commit();
        tma_wait_read<0>();
    }
}

}  // namespace tdx
