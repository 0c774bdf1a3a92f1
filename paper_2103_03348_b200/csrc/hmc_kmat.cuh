// hmc_kmat.cuh -- the "cached kernel matrix" evaluation of the z-posterior inside one hawkes_hmc_run call (included
// by hawkes.cu inside its anonymous namespace).
//
// Inside one call only the M sequenced rates theta_m = exp(z_m + beta t_m) change; events, hyperparameters and the
// other rates (= 1) are fixed.  Therefore, with K[n][k] = exp(-omega (t_n - t_m) - |x_n - x_m|^2 / 2h^2) I[t_m < t_n]
// for m = idx[k] (N x M doubles, 302 MB at N = 23,422, M = 1,610; built once per call) and
// lambda0_n = (background sum) + CS sum_{m not sequenced} k-terms (one ordinary pass 1 with the sequenced rates set to 0),
//   lambda_n = lambda0_n + CS sum_k K[n][k] theta_k           (row sums:    one pass over K)
//   c_k      = sum_n K[n][k] / lambda_n,  d_k = sum_n (K[n][k] / lambda_n)^2   (column sums: one pass over K)
// are the same sums as Eq. 1 / Eq. 4 / Eq. 5 of the paper with the pair terms cached: HBM-bound (two reads of K per
// evaluation) instead of FP64-bound.  It is not the paper's method (which recomputes every pair) and is
// reported as a separate variant.  All sums in fixed order.

constexpr int KM_ROWS_T = 256;      // kmat_rows_kernel: 8 warps = 8 rows per CTA

__global__ void kmat_build_kernel(const double* __restrict__ rec, int64_t n, int64_t m, const int64_t* __restrict__ idx,
                                  double omega, double inv_2h2, double* __restrict__ K) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n * m) return;
    const int64_t i = e / m, k = e - i * m;
    const double4 a = reinterpret_cast<const double4*>(rec)[i];          // (x, y, t, .): dim <= 2 records
    const double4 b = reinterpret_cast<const double4*>(rec)[idx[k]];
    const double dt = a.z - b.z, dx = a.x - b.x, dy = a.y - b.y;
    K[e] = dt > 0.0 ? exp(-omega * dt - (dx * dx + dy * dy) * inv_2h2) : 0.0;
}

// theta_k = exp(z_k + beta t_k), E-terms of the integral: thM[k], and per-CTA partial of sum_k theta_k (1 - E_k)
__global__ void kmat_theta_kernel(int64_t m, const int64_t* __restrict__ idx, const double* __restrict__ z, double beta,
                                  const double* __restrict__ t, double* __restrict__ thM) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < m) thM[k] = exp(z[k] + beta * t[idx[k]]);
}

// rows: lambda_n = lambda0_n + CS sum_k K[n][k] theta_k; w_n = 1 / lambda_n; CTA partial of sum log lambda_n
__global__ void __launch_bounds__(KM_ROWS_T) kmat_rows_kernel(const double* __restrict__ K, int64_t n, int64_t m,
                                                              const double* __restrict__ thM, const double* __restrict__ lam0,
                                                              double CS, double* __restrict__ w, double* __restrict__ logpart,
                                                              unsigned* __restrict__ status) {
    extern __shared__ double sth[];
    __shared__ double wl[KM_ROWS_T / 32];
    for (int64_t k = threadIdx.x; k < m; k += KM_ROWS_T) sth[k] = thM[k];
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t row = (int64_t)blockIdx.x * (KM_ROWS_T / 32) + wid;
    double ll = 0.0;
    if (row < n) {
        const double* kr = K + row * m;
        double s = 0.0;
        for (int64_t k = lane; k < m; k += 32) s = fma(kr[k], sth[k], s);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
        if (lane == 0) {
            const double L = fma(CS, s, lam0[row]);
            w[row] = 1.0 / L;
            ll = log(L);
            if (L == 0.0) atomicOr(status, (unsigned)ST_ZERO_RATE);
        }
    }
    if (lane == 0) wl[wid] = ll;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int q = 0; q < KM_ROWS_T / 32; ++q) a += wl[q];
        logpart[blockIdx.x] = a;
    }
}

// columns: CTA (bx, by) owns columns [256 bx, 256 bx + 256) and rows [by rows_per, (by+1) rows_per); one column per
// thread, rows in order (eight loads in flight): partial[by][k] (c) and partial[nby + by][k] (d, when want_d)
constexpr int KM_COL_TILE = 256;
__global__ void __launch_bounds__(KM_COL_TILE) kmat_cols_kernel(const double* __restrict__ K, int64_t n, int64_t m,
                                                                const double* __restrict__ w, int rows_per, int want_d,
                                                                double* __restrict__ part) {
    const int64_t k = (int64_t)blockIdx.x * KM_COL_TILE + threadIdx.x;
    const int64_t r0 = (int64_t)blockIdx.y * rows_per, r1 = min(r0 + rows_per, n);
    if (k >= m) return;
    double c = 0.0, d = 0.0;
    int64_t i = r0;
    for (; i + 8 <= r1; i += 8) {
        double q[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) q[u] = K[(i + u) * m + k];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const double v = q[u] * w[i + u];
            c += v;
            d = fma(v, v, d);
        }
    }
    for (; i < r1; ++i) {
        const double v = K[i * m + k] * w[i];
        c += v;
        d = fma(v, v, d);
    }
    part[(int64_t)blockIdx.y * m + k] = c;
    if (want_d) part[((int64_t)gridDim.y + blockIdx.y) * m + k] = d;
}

// finish: one warp per column adds the row-block partials (lane l takes blocks l, l + 32, ... in order, then a fixed
// shuffle tree); d ell/d theta_k = CS c_k - xi0 (1 - E_k); chain rule to z; CTA partial of sum_k theta_k (1 - E_k)
__global__ void __launch_bounds__(256) kmat_finish_kernel(int64_t m, int nblk_c, const double* __restrict__ part, int want_d,
                                   const int64_t* __restrict__ idx, const double* __restrict__ t, int64_t n,
                                   const double* __restrict__ thM, double CS, double xi0, double omega,
                                   const double* __restrict__ prior_grad, double* __restrict__ grad_z,
                                   double* __restrict__ hess_z, double* __restrict__ intpart) {
    __shared__ double sm[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * 8 + wid;
    double ti = 0.0;
    if (k < m) {
        double c = 0.0, d = 0.0;
        for (int b = lane; b < nblk_c; b += 32) c += part[(int64_t)b * m + k];
        if (want_d)
            for (int b = lane; b < nblk_c; b += 32) d += part[((int64_t)nblk_c + b) * m + k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            c += __shfl_down_sync(0xffffffffu, c, off);
            d += __shfl_down_sync(0xffffffffu, d, off);
        }
        if (lane == 0) {
            const double th = thM[k], one_minus_E = -expm1(-omega * (t[n - 1] - t[idx[k]]));
            const double g = th * (CS * c - xi0 * one_minus_E);
            if (grad_z) grad_z[k] = prior_grad ? g + prior_grad[k] : g;
            if (hess_z) hess_z[k] = fma(th * th, -(CS * CS) * d, g);
            ti = th * one_minus_E;
        }
    }
    if (lane == 0) sm[wid] = ti;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int q = 0; q < 8; ++q) a += sm[q];
        intpart[blockIdx.x] = a;
    }
}

// ell = sum log lambda - (Lambda0 + xi0 sum_k theta_k (1 - E_k)); out3 = (ell, log prior, sum).  One warp: lane l adds
// entries l, l + 32, ... in order, then a fixed shuffle tree.
__global__ void kmat_scalar_kernel(int nblk_r, const double* __restrict__ logpart, int nblk_f, const double* __restrict__ intpart,
                                   const double* __restrict__ lam0_integral, double xi0, const double* __restrict__ logprior,
                                   double* __restrict__ out3) {
    const int lane = threadIdx.x;
    double sl = 0.0, si = 0.0;
    for (int b = lane; b < nblk_r; b += 32) sl += logpart[b];
    for (int b = lane; b < nblk_f; b += 32) si += intpart[b];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sl += __shfl_down_sync(0xffffffffu, sl, off);
        si += __shfl_down_sync(0xffffffffu, si, off);
    }
    if (lane == 0) {
        const double ell = sl - (lam0_integral[0] + xi0 * si);
        out3[0] = ell;
        out3[1] = logprior[0];
        out3[2] = ell + logprior[0];
    }
}

// theta = 1 everywhere except the sequenced events, which get 0 (set-up evaluation of lambda0)
__global__ void kmat_zero_scatter_kernel(int64_t m, const int64_t* __restrict__ idx, double* __restrict__ theta) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < m) theta[idx[k]] = 0.0;
}

// ------------------------------------------------------------------------------------------------
// Dense Hessian block of the sequenced rates (hawkes_hessian_theta_block): A[n][k] = CS K[n][k] / lambda_n, then
// H = -A^T A, M x M.  A contraction over n, written as a plain tiled fp64 kernel (64 x 64 output tile per CTA, 4 x 4
// per thread, 16 rows of A per shared-memory stage); only tiles on or above the diagonal are computed, the mirror
// image is written with them.  Not on the hot path; untuned.
__global__ void kmat_scale_rows_kernel(int64_t n, int64_t m, double CS, const double* __restrict__ lam,
                                       double* __restrict__ A) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n * m) return;
    A[e] = CS * A[e] / lam[e / m];
}

constexpr int HB_TILE = 64, HB_ROWS = 16;
__global__ void __launch_bounds__(256) hess_block_kernel(const double* __restrict__ A, int64_t n, int64_t m,
                                                         double* __restrict__ H) {
    if (blockIdx.x < blockIdx.y) return;                      // tiles on or above the diagonal only
    __shared__ double sa[HB_ROWS][HB_TILE], sb[HB_ROWS][HB_TILE];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const int64_t k0 = (int64_t)blockIdx.y * HB_TILE, l0 = (int64_t)blockIdx.x * HB_TILE;
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    for (int64_t r0 = 0; r0 < n; r0 += HB_ROWS) {
        for (int q = threadIdx.x; q < HB_ROWS * HB_TILE; q += 256) {
            const int rr = q / HB_TILE, cc = q % HB_TILE;
            const int64_t r = r0 + rr;
            sa[rr][cc] = (r < n && k0 + cc < m) ? A[r * m + k0 + cc] : 0.0;
            sb[rr][cc] = (r < n && l0 + cc < m) ? A[r * m + l0 + cc] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int rr = 0; rr < HB_ROWS; ++rr) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { a[i] = sa[rr][ty * 4 + i]; b[i] = sb[rr][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t k = k0 + ty * 4 + i, l = l0 + tx * 4 + j;
            if (k < m && l < m) {
                H[k * m + l] = -acc[i][j];
                H[l * m + k] = -acc[i][j];
            }
        }
}
