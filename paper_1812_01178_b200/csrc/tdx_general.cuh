// tdx_general.cuh -- batched tridiagonal solve with PER-LINE coefficients and diagonal pivoting.
// for the y-solves of the Poisson equation "a parallel tridiagonal solver with diagonal pivoting is used
// [3]" because those systems are only weakly dominant (L172).  This is that role for systems that are not dominant at
// all: every line brings its own a, b, c (three more field-sized arrays, +24 B per value -- SURVEY 8(d) counts it), and
// the elimination chooses 1x1 or 2x2 diagonal pivots without row interchanges (the criterion of the diagonal-pivoting
// family [3] builds on: with sigma = max(|c_i|, |a_{i+1}|, |b_{i+1}|, |c_{i+1}|, |a_{i+2}|) take the 1x1 pivot b_i when
// |b_i| sigma >= kappa |c_i a_{i+1}|, kappa = (sqrt 5 - 1)/2, else the 2x2 block of rows i, i+1).
//
// Thread = line (lines of y or z: adjacent threads are adjacent x, so every access is coalesced); all lanes of a warp
// walk the rows in lockstep -- a lane whose row is the second row of a 2x2 pivot idles for that row -- so a rolling
// three-row window in registers loads every coefficient exactly once.  Two passes over HBM (this is the pivoting
// BASELINE, the counterpart of k_thomas_strided, not a partition method): forward writes the modified diagonal, the
// modified right-hand side and the pivot type; backward substitutes in place.
#pragma once
#include <cuda_runtime.h>

namespace tdx {

// a, b, c, d: [outer][n][inner] with inner contiguous (line stride = inner); bm: modified diagonal (same shape);
// flag: bytes, same shape: 0 = 1x1 pivot row, 1 = first row of a 2x2 pivot, 2 = second row.
template <bool PIVOT>
__global__ void __launch_bounds__(128) k_general_forward(const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ c,
                                                         double* __restrict__ d, double* __restrict__ bm, unsigned char* __restrict__ flag,
                                                         int n, long long inner, long long outer) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= inner) return;
    const size_t base = (size_t)blockIdx.y * n * inner + i;
    const double kappa = 0.6180339887498949;
    // window rows r0 = j, r1 = j+1, r2 = j+2; rows past the end are identity rows (a = c = d = 0, b = 1)
    double b0 = b[base], c0 = (n > 1) ? c[base] : 0.0, d0 = d[base];
    double a1 = 0.0, b1 = 1.0, c1 = 0.0, d1 = 0.0, a2 = 0.0, b2 = 1.0, c2 = 0.0, d2 = 0.0;
    if (n > 1) { const size_t q = base + inner; a1 = a[q]; b1 = b[q]; c1 = (n > 2) ? c[q] : 0.0; d1 = d[q]; }
    if (n > 2) { const size_t q = base + 2 * inner; a2 = a[q]; b2 = b[q]; c2 = (n > 3) ? c[q] : 0.0; d2 = d[q]; }
    bool second = false;
    for (int j = 0; j < n; ++j) {
        unsigned char fl = 0;
        if (second) {
            fl = 2; second = false;
        } else {
            bool one = true;
            if (PIVOT) {
                const double sigma = fmax(fmax(fabs(c0), fabs(a1)), fmax(fabs(b1), fmax(fabs(c1), fabs(a2))));
                one = fabs(b0) * sigma >= kappa * fabs(c0 * a1);
            }
            if (one) {
                const double m = a1 / b0;
                b1 = fma(-m, c0, b1);
                d1 = fma(-m, d0, d1);
            } else {
                fl = 1; second = true;
                const double idet = 1.0 / (b0 * b1 - a1 * c0);
                b2 = fma(-a2 * idet, b0 * c1, b2);
                d2 = fma(-a2 * idet, b0 * d1 - a1 * d0, d2);
            }
        }
        const size_t q = base + (size_t)j * inner;
        bm[q] = b0; d[q] = d0; flag[q] = fl;
        b0 = b1; c0 = c1; d0 = d1;
        a1 = a2; b1 = b2; c1 = c2; d1 = d2;
        if (j + 3 < n) { const size_t q3 = base + (size_t)(j + 3) * inner; a2 = a[q3]; b2 = b[q3]; c2 = (j + 4 < n) ? c[q3] : 0.0; d2 = d[q3]; }
        else { a2 = 0.0; b2 = 1.0; c2 = 0.0; d2 = 0.0; }
    }
}

__global__ void __launch_bounds__(128) k_general_backward(const double* __restrict__ a, const double* __restrict__ c, double* __restrict__ d,
                                                          const double* __restrict__ bm, const unsigned char* __restrict__ flag,
                                                          int n, long long inner, long long outer) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= inner) return;
    const size_t base = (size_t)blockIdx.y * n * inner + i;
    double xn = 0.0, pending = 0.0;                                   // x_{j+1}; x_j computed one row early by a 2x2 pivot
    for (int j = n - 1; j >= 0; --j) {
        const size_t q = base + (size_t)j * inner;
        const unsigned char fl = flag[q];
        double x;
        if (fl == 0) {
            const double cj = (j < n - 1) ? c[q] : 0.0;
            x = (d[q] - cj * xn) / bm[q];
        } else if (fl == 2) {                                         // rows j-1, j: [[b0, c0],[a1, b1]] (x_{j-1}, x_j) = (d_{j-1}, d_j - c_j x_{j+1})
            const size_t p = q - inner;
            const double b0 = bm[p], c0 = c[p], a1 = a[q], b1 = bm[q];
            const double cj = (j < n - 1) ? c[q] : 0.0;
            const double r1 = d[p], r2 = d[q] - cj * xn;
            const double idet = 1.0 / (b0 * b1 - a1 * c0);
            x = (b0 * r2 - a1 * r1) * idet;
            pending = (b1 * r1 - c0 * r2) * idet;
        } else {
            x = pending;
        }
        d[q] = x;
        xn = x;
    }
}

}  // namespace tdx
