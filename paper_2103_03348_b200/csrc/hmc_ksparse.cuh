// hmc_ksparse.cuh -- the cached kernel matrix of hmc_kmat.cuh with its exact zeros left out (included by hawkes.cu
// inside its anonymous namespace; DESIGN.md sections 12 and 13).
//
// K[n][k] = exp(-omega (t_n - t_m) - |x_n - x_m|^2 / 2h^2) I[t_m < t_n], m = idx[k], is exactly +0.0 for every pair that
// is acausal or further apart than the kernel reaches in fp64 (section 13): at configs[3] all but a fraction of a
// percent of its N x M entries.  After the dense build (once per hawkes_hmc_run call) the non-zeros are compressed
// twice, by row (for lambda_n = lambda0_n + CS sum_k K[n][k] theta_k) and by column (for c_k = sum_n K[n][k] / lambda_n
// and d_k), each in index order, so that an evaluation reads a few MB instead of 2 x 302 MB.  Every sum keeps a fixed
// order (lane l takes entries l, l + 32, ... of its row or column, then a fixed shuffle tree): bit-identical run to run.
// Only exact zeros are dropped: the values are those of the dense cached-matrix variant in another summation order.

constexpr int KS_ROWS_PER = 512;    // rows per CTA row-block of the column compression

// entries != 0 of every row (one warp per row, 8 rows per CTA); cnt[n] = 0 closes the array for the exclusive scan
__global__ void __launch_bounds__(256) ksp_row_count_kernel(const double* __restrict__ K, int64_t n, int64_t m,
                                                            int64_t* __restrict__ cnt) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t row = (int64_t)blockIdx.x * 8 + wid;
    if (row > n) return;
    if (row == n) { if (lane == 0) cnt[n] = 0; return; }
    const double* kr = K + row * m;
    int c = 0;
    for (int64_t k = lane; k < m; k += 32) c += kr[k] != 0.0 ? 1 : 0;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
    if (lane == 0) cnt[row] = c;
}

// the row's non-zeros in column order at rowptr[row] ..
__global__ void __launch_bounds__(256) ksp_row_fill_kernel(const double* __restrict__ K, int64_t n, int64_t m,
                                                           const int64_t* __restrict__ rowptr, int* __restrict__ col,
                                                           double* __restrict__ val) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t row = (int64_t)blockIdx.x * 8 + wid;
    if (row >= n) return;
    const double* kr = K + row * m;
    int64_t base = rowptr[row];
    for (int64_t k0 = 0; k0 < m; k0 += 32) {
        const int64_t k = k0 + lane;
        const double v = k < m ? kr[k] : 0.0;
        const unsigned b = __ballot_sync(0xffffffffu, v != 0.0);
        if (v != 0.0) {
            const int64_t pos = base + __popc(b & ((1u << lane) - 1u));
            col[pos] = (int)k;
            val[pos] = v;
        }
        base += __popc(b);
    }
}

// columns: CTA (bx, by) counts the non-zeros of columns [256 bx, +256) in rows [by KS_ROWS_PER, +KS_ROWS_PER)
__global__ void __launch_bounds__(256) ksp_col_count_kernel(const double* __restrict__ K, int64_t n, int64_t m,
                                                            int* __restrict__ cntc) {
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= m) return;
    const int64_t r0 = (int64_t)blockIdx.y * KS_ROWS_PER, r1 = min(r0 + KS_ROWS_PER, n);
    int c = 0;
    for (int64_t i = r0; i < r1; ++i) c += K[i * m + k] != 0.0 ? 1 : 0;
    cntc[(int64_t)blockIdx.y * m + k] = c;
}

// one CTA: column totals -> colptr (serial scan over the m columns), then the offset of every (row block, column)
__global__ void __launch_bounds__(1024) ksp_col_offsets_kernel(int nrb, int64_t m, const int* __restrict__ cntc,
                                                               int64_t* __restrict__ colptr, int64_t* __restrict__ offc) {
    for (int64_t k = threadIdx.x; k < m; k += blockDim.x) {
        int64_t tot = 0;
        for (int b = 0; b < nrb; ++b) tot += cntc[(int64_t)b * m + k];
        colptr[k + 1] = tot;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t run = 0;
        colptr[0] = 0;
        for (int64_t k = 0; k < m; ++k) { run += colptr[k + 1]; colptr[k + 1] = run; }
    }
    __syncthreads();
    for (int64_t k = threadIdx.x; k < m; k += blockDim.x) {
        int64_t run = colptr[k];
        for (int b = 0; b < nrb; ++b) { offc[(int64_t)b * m + k] = run; run += cntc[(int64_t)b * m + k]; }
    }
}

__global__ void __launch_bounds__(256) ksp_col_fill_kernel(const double* __restrict__ K, int64_t n, int64_t m,
                                                           const int64_t* __restrict__ offc, int* __restrict__ rowi,
                                                           double* __restrict__ valc) {
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= m) return;
    const int64_t r0 = (int64_t)blockIdx.y * KS_ROWS_PER, r1 = min(r0 + KS_ROWS_PER, n);
    int64_t pos = offc[(int64_t)blockIdx.y * m + k];
    for (int64_t i = r0; i < r1; ++i) {
        const double v = K[i * m + k];
        if (v != 0.0) { rowi[pos] = (int)i; valc[pos] = v; ++pos; }
    }
}

// rows: lambda_n = lambda0_n + CS sum_j val[j] theta[col[j]]; w_n = 1 / lambda_n; CTA partial of sum log lambda_n
// (outputs as kmat_rows_kernel)
__global__ void __launch_bounds__(KM_ROWS_T) ksp_rows_kernel(const int64_t* __restrict__ rowptr, const int* __restrict__ col,
                                                             const double* __restrict__ val, int64_t n,
                                                             const double* __restrict__ thM, const double* __restrict__ lam0,
                                                             double CS, double* __restrict__ w, double* __restrict__ logpart,
                                                             unsigned* __restrict__ status) {
    __shared__ double wl[KM_ROWS_T / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t row = (int64_t)blockIdx.x * (KM_ROWS_T / 32) + wid;
    double ll = 0.0;
    if (row < n) {
        double s = 0.0;
        const int64_t j1 = rowptr[row + 1];
        for (int64_t j = rowptr[row] + lane; j < j1; j += 32) s = fma(val[j], thM[col[j]], s);
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

// columns: one warp per column; part[k] = c_k, part[m + k] = d_k: the layout kmat_finish_kernel reads with one row block
__global__ void __launch_bounds__(256) ksp_cols_kernel(const int64_t* __restrict__ colptr, const int* __restrict__ rowi,
                                                       const double* __restrict__ valc, int64_t m,
                                                       const double* __restrict__ w, int want_d, double* __restrict__ part) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * 8 + wid;
    if (k >= m) return;
    double c = 0.0, d = 0.0;
    const int64_t j1 = colptr[k + 1];
    for (int64_t j = colptr[k] + lane; j < j1; j += 32) {
        const double v = valc[j] * w[rowi[j]];
        c += v;
        d = fma(v, v, d);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        c += __shfl_down_sync(0xffffffffu, c, off);
        d += __shfl_down_sync(0xffffffffu, d, off);
    }
    if (lane == 0) {
        part[k] = c;
        if (want_d) part[m + k] = d;
    }
}
