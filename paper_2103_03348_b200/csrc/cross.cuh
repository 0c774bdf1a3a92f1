// cross.cuh -- the N x 6 block d2 ell / d theta_m dp of the Hessian (BASELINE.json configs[0]
// "full gradient and Hessian"), as a third pairwise pass on the decomposition of pass 2.  Included by hawkes.cu inside
// its anonymous namespace, after pass2_kernel.
//
//   d2 ell / d theta_m dp = sum_{n: t_n > t_m} k_nm [ (d log k_nm / dp) / lambda_n - lambda_{n,p} / lambda_n^2 ] - d2 Lambda / d theta_m dp
//
// (Eq. 4, differentiated once more; d log k / d(xi0, h, omega) = (1/xi0, r^2/h^3 - D/h, 1/omega - dt), zero for
// the background's three; d2 Lambda / d theta_m d xi0 = 1 - E_m, d2 Lambda / d theta_m d omega = xi0 T_m E_m.)  With
// a_nm = k_nm / lambda_n and rho_{n,p} = lambda_{n,p} / lambda_n the source m needs nine sums over its later targets,
//
//   A = sum a,   A_r = sum a r^2,   A_t = sum a dt,   X_p = sum a rho_{n,p}  (p = 0..5),
//
// and  cross[m] = ( -X_0, -X_1, -X_2,  A/xi0 - X_3 - (1 - E_m),  A_r/h^3 - D A/h - X_4,  A/omega - A_t - X_5 - xi0 T_m E_m ).
//
// The thread owns R sources (nine accumulators each); the targets stream through shared memory as records of
// RS + 6 doubles, (x, y, [z,] t, 1/lambda_n, [0,] rho_0..rho_5), which reduce1 writes when the block is wanted.  Same
// stream-K split (`tri` form), same partial-slot layout and fixed-order reduction as pass 2: bit-identical run to run.

constexpr int XM = 9;   // moments per source

template <bool DIM3> constexpr int cross_rs() { return (DIM3 ? 6 : 4) + 6; }
template <bool DIM3> constexpr unsigned cross_group_bytes() { return 2u * TS * cross_rs<DIM3>() * sizeof(double); }

// streamed tile of TS records of RSX doubles, double-buffered through registers (as RecIO)
template <int RSX>
struct TileIO {
    static constexpr int CH = RSX / 2;
    static constexpr int PER_THREAD = TS * CH / NT;
    double2 v[PER_THREAD];
    __device__ __forceinline__ void load(const double* __restrict__ src, int64_t first, int cnt, int tid) {
        const double2* g = reinterpret_cast<const double2*>(src) + first * CH;
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int c = tid + q * NT;
            v[q] = (c < cnt * CH) ? __ldg(g + c) : make_double2(0.0, 0.0);
        }
    }
    __device__ __forceinline__ void store(double* buf, int tid) const {
        double2* s = reinterpret_cast<double2*>(buf);
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) s[tid + q * NT] = v[q];
    }
};

template <int R, bool MASKED, bool DIM3>
__device__ __forceinline__ void cross_tile(const double* __restrict__ sbuf, int cnt, const Ev<DIM3> (&g)[R],
                                           double (&acc)[R][XM], const P1C& c, unsigned lane_base) {
    constexpr int RS = DIM3 ? 6 : 4;
    constexpr int RSX = cross_rs<DIM3>();
#pragma unroll 2
    for (int j = 0; j < cnt; ++j) {
        const double* rp = sbuf + j * RSX;
        const Ev<DIM3> s = read_rec<DIM3>(rp);   // a target; s.w = 1/lambda_n
        double rho[6];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double2 v = reinterpret_cast<const double2*>(rp + RS)[k];
            rho[2 * k] = v.x;
            rho[2 * k + 1] = v.y;
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double dx = s.x - g[r].x, dy = s.y - g[r].y, dt = s.t - g[r].t;
            double u = fma(dy, dy, dx * dx);
            if (DIM3) { const double dz = s.z - g[r].z; u = fma(dz, dz, u); }
            const double as = fma(c.rho_s, dt, u);
            const double e = exp2_scaled<MASKED ? 2 : 0>(as, c.negcs, c.lim_s_hi, dt, c.e, lane_base);
            // an acausal pair is no term of the sums: it must add exactly 0 even when 1/lambda_n = inf
            const bool live = !MASKED || dt > 0.0;
            const double q = live ? e * s.w : 0.0;
            acc[r][0] += q;
            acc[r][1] = fma(q, u, acc[r][1]);
            acc[r][2] = fma(q, live ? dt : 0.0, acc[r][2]);
#pragma unroll
            for (int p = 0; p < 6; ++p) acc[r][3 + p] = fma(q, live ? rho[p] : 0.0, acc[r][3 + p]);
        }
    }
}

// partx[(slot*XM + k)*ld + m]
template <int R, bool DIM3, int G>
__global__ void __launch_bounds__(NT * G, 1) cross_pass_kernel(const double* __restrict__ rec, const double* __restrict__ crec,
                                                               int64_t n, int64_t ld, DevConsts c,
                                                               const double* __restrict__ tab_g, double* __restrict__ partx,
                                                               Split sp) {
    constexpr int RS = DIM3 ? 6 : 4;
    constexpr int RSX = cross_rs<DIM3>();
    constexpr int TOFF = DIM3 ? 3 : 2;
    constexpr unsigned BUF = cross_group_bytes<DIM3>();
    static_assert(smem_request(G * BUF) <= SMEM_MAX, "table + streaming buffers must fit shared memory");
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double smagic;
    const unsigned smem_base = (unsigned)__cvta_generic_to_shared(smem);
    const SmemPlan plan = smem_plan(smem_base, G * BUF);
    fill_table(reinterpret_cast<double*>(smem + plan.tab_off), tab_g);
    stash_consts(smagic);
    __syncthreads();

    const int grp = threadIdx.x / NT, tid = threadIdx.x % NT;
    const int64_t vcta = (int64_t)blockIdx.x * G + grp + sp.w_begin;
    double* const sbuf0 = reinterpret_cast<double*>(smem + plan.buf_off + grp * BUF);
    double* const sbuf1 = sbuf0 + TS * RSX;
    const unsigned lane_base = (smem_base + plan.tab_off) | (8u * (threadIdx.x & 31));

    const int64_t total = split_prefix(sp, sp.n_tiles);
    const int64_t lo = vcta * sp.chunk;
    if (lo >= total || vcta >= sp.w_end) return;
    const int64_t hi = min(lo + sp.chunk, total);
    const P1C pc = pinned_consts(smagic, c);

    for (int M = split_tile_of(sp, lo); M < sp.n_tiles; ++M) {
        const int64_t base = split_prefix(sp, M);
        if (base >= hi) break;
        const int64_t cost_M = split_prefix(sp, M + 1) - base;
        const int64_t jb = split_pos(sp, M, max(lo - base, (int64_t)0));
        const int64_t je = split_pos(sp, M, min(hi - base, cost_M));
        const int64_t m0 = (int64_t)M * (NT * R);
        const int64_t m1 = min(m0 + (int64_t)NT * R, n);

        Ev<DIM3> g[R];
        double acc[R][XM];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = min(m0 + r * NT + tid, n - 1);
            g[r] = read_rec<DIM3>(rec + i * RS);
#pragma unroll
            for (int k = 0; k < XM; ++k) acc[r][k] = 0.0;
        }
        const double t_last = rec[(m1 - 1) * RS + TOFF];   // latest own source time

        // a piece is "plain" when every pair in it is causal (all targets after the tile, no tie across the boundary)
        auto is_plain = [&](int64_t a_) { return a_ >= m1 && crec[a_ * RSX + TOFF] > t_last; };
        TileIO<RSX> io;
        int64_t a = jb;
        int64_t b = min(je, (a / TS + 1) * TS);
        group_sync(grp);
        if (a < je) {
            io.load(crec, a, (int)(b - a), tid);
            io.store(sbuf0, tid);
        }
        group_sync(grp);
        int cur = 0;
        while (a < je) {
            const int cnt = (int)(b - a);
            const int64_t a2 = b, b2 = min(je, b + TS);
            if (a2 < je) io.load(crec, a2, (int)(b2 - a2), tid);
            const double* sb = cur ? sbuf1 : sbuf0;
            if (is_plain(a)) cross_tile<R, false, DIM3>(sb, cnt, g, acc, pc, lane_base);
            else cross_tile<R, true, DIM3>(sb, cnt, g, acc, pc, lane_base);
            if (a2 < je) io.store(cur ? sbuf0 : sbuf1, tid);
            group_sync(grp);
            cur ^= 1;
            a = a2;
            b = b2;
        }
        const int slot = split_slot_of(sp, vcta, base);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = m0 + r * NT + tid;
            if (i < n) {
#pragma unroll
                for (int k = 0; k < XM; ++k) partx[(int64_t)(slot * XM + k) * ld + i] = acc[r][k];
            }
        }
    }
}

// fixed-order sum of the partial slots and the closed-form terms: cross[m*6 + p]
template <bool DIM3>
__global__ void __launch_bounds__(RED_T) cross_finish_kernel(const double* __restrict__ rec, int64_t n, int64_t ld, DevConsts c,
                                                             const double* __restrict__ partx, Split sp,
                                                             double* __restrict__ cross) {
    constexpr int RS = DIM3 ? 6 : 4;
    const int64_t i = (int64_t)blockIdx.x * RED_T + threadIdx.x;
    if (i >= n) return;
    double s[XM];
#pragma unroll
    for (int k = 0; k < XM; ++k) s[k] = 0.0;
    int slot0, n_slots;
    split_slots(sp, i / sp.tile, &slot0, &n_slots);
    for (int q = 0; q < n_slots; ++q) {
        double v[XM];
#pragma unroll
        for (int k = 0; k < XM; ++k) v[k] = partx[(int64_t)(q * XM + k) * ld + i];
#pragma unroll
        for (int k = 0; k < XM; ++k) s[k] += v[k];
    }
    const double D = (double)c.dim;
    const double tN = rec[(n - 1) * RS + (DIM3 ? 3 : 2)];
    const double T = tN - rec[i * RS + (DIM3 ? 3 : 2)];
    const double A = c.CSS * s[0], Ar = c.CSS * s[1], At = c.CSS * s[2];
    double X[6];
#pragma unroll
    for (int p = 0; p < 6; ++p) X[p] = c.CSS * s[3 + p];
    double* o = cross + i * 6;
    o[0] = -X[0];
    o[1] = -X[1];
    o[2] = -X[2];
    o[3] = A / c.xi0 - X[3] - (-expm1(-c.omega * T));
    o[4] = Ar / (c.h * c.h * c.h) - D * A / c.h - X[4];
    o[5] = A / c.omega - At - X[5] - c.xi0 * T * exp(-c.omega * T);
}
