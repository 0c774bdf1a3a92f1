// shard.cuh -- one evaluation sharded across `world` GPUs.
// Included by hawkes.cu after its kernels, the context and enqueue helpers.
//
// Every rank holds all events (32 B each).  The cost axis of a pairwise pass (Split, hawkes.cu) is cut into
// world x W equal chunks instead of W, and rank r runs the workers [r W, (r+1) W) of that cut: a contiguous range of
// the axis, so the ranks' loads are equal by construction whatever the triangle looks like.  What a rank computes is
// a PARTIAL sum for every event its range touches (row sums of its target tiles, column sums of the background for the
// events it streamed); the partial sums of all ranks are exchanged once per pass and added in rank order:
//
//   phase A  hawkes_shard_pass1    prep + pass 1 over the rank's workers -> per-event partial moment sums  [NM][ld]
//   exchange all-gather of the NM x ld doubles (NCCL; the binding does it)
//   phase B  hawkes_shard_reduce1  sum over ranks in rank order, lambda_n, 1/lambda_n, the O(N) scalar sums -> ell, grad_hyper,
//                                  hess_hyper: computed by every rank from the same numbers in the same order (replicated,
//                                  bit-identical across ranks), so the scalars need no second collective
//   phase C  hawkes_shard_pass2    pass 2 over the rank's workers -> partial (c_m, d_m)                     [2][ld]
//   exchange all-gather of the 2 x ld doubles
//   phase D  hawkes_shard_finish   sum over ranks in rank order -> grad_theta, hess_theta_diag (replicated)
//
// Fixed cut + fixed rank order => bit-identical results run to run for a given `world` (they differ from the one-GPU
// result by summation order alone).  The kernels of the phases are the ones of the one-GPU path: a Split carries the
// worker range of the launch, and the gathered per-rank sums are read by reduce1_kernel / theta_kernel as `world`
// partial slots per tile.

// partial sums of one rank: out[k*ld + i], k < 2 NB (b moments, then s moments); the b sums hold the rank's row
// partials and, for the symmetric pass 1, its column partials of event i (tiles in index order)
template <int LEVEL>
__global__ void __launch_bounds__(RED_T) shard_sum1_kernel(int64_t n, int64_t ld, const double* __restrict__ part, Split sp,
                                                           const double* __restrict__ partc, int sym_tile,
                                                           double* __restrict__ out) {
    constexpr int NB = Mom<LEVEL>::NB;
    const int64_t i = (int64_t)blockIdx.x * RED_T + threadIdx.x;
    if (i >= n) return;
    double b[NB], s[NB];
#pragma unroll
    for (int k = 0; k < NB; ++k) { b[k] = 0.0; s[k] = 0.0; }
    int slot0, n_slots;
    split_slots(sp, i / sp.tile, &slot0, &n_slots);
    for (int q = 0; q < n_slots; ++q) {
        const double* o = part + (int64_t)q * (2 * NB) * ld + i;
#pragma unroll
        for (int k = 0; k < NB; ++k) { b[k] += o[(int64_t)k * ld]; s[k] += o[(int64_t)(NB + k) * ld]; }
    }
    if (partc != nullptr) {
        // column partial (tile I, event i) was written by this rank iff i lies in the range of tile I's streamed events
        // that the rank's workers covered
        const int64_t total = split_prefix(sp, sp.n_tiles);
        const int64_t lo = (int64_t)sp.w_begin * sp.chunk;
        int64_t hi = (int64_t)sp.w_end * sp.chunk;
        if (hi > total) hi = total;
        if (lo < hi) {
            const int Ia = split_tile_of(sp, lo), Ib = split_tile_of(sp, hi - 1);
            int I = (int)(i / sym_tile);
            if (I < Ia) I = Ia;
            for (; I <= Ib; ++I) {
                if (I == Ia || I == Ib) {
                    const int64_t base = split_prefix(sp, I), cost_I = split_prefix(sp, I + 1) - base;
                    const int64_t jb = split_pos(sp, I, lo > base ? lo - base : 0);
                    const int64_t je = split_pos(sp, I, hi - base < cost_I ? hi - base : cost_I);
                    if (i < jb || i >= je) continue;
                }
                const int sc = I - (int)(i / sym_tile);
#pragma unroll
                for (int k = 0; k < NB; ++k) b[k] += partc[colpart_index(sp.n_tiles, sym_tile, NB, sc, k, i)];
            }
        }
    }
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        out[(int64_t)k * ld + i] = b[k];
        out[(int64_t)(NB + k) * ld + i] = s[k];
    }
}

__global__ void __launch_bounds__(RED_T) shard_sum2_kernel(int64_t n, int64_t ld, const double* __restrict__ part2, Split sp,
                                                           int with_d, double* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * RED_T + threadIdx.x;
    if (i >= n) return;
    double cs = 0.0, ds = 0.0;
    int slot0, n_slots;
    split_slots(sp, i / sp.tile, &slot0, &n_slots);
    for (int q = 0; q < n_slots; ++q) {
        cs += part2[(int64_t)(q * 2 + 0) * ld + i];
        if (with_d) ds += part2[(int64_t)(q * 2 + 1) * ld + i];
    }
    out[i] = cs;
    out[ld + i] = ds;
}

struct ShardLevels { int level1, level2, sym; };
inline ShardLevels shard_levels(const hawkes_ctx* ctx, uint32_t want) {
    ShardLevels L;
    L.level1 = (want & HAWKES_WANT_HESS_HYPER) ? 2 : ((want & HAWKES_WANT_GRAD_HYPER) ? 1 : 0);
    L.level2 = (want & HAWKES_WANT_HESS_THETA) ? 1 : 0;
    L.sym = (ctx->d_partc != nullptr && L.level1 <= 1 && !ctx->force_dense) ? 1 : 0;
    return L;
}

// the cut of both passes for (n, want, world): the same on every rank
inline void shard_plan(const hawkes_ctx* ctx, int64_t n, const ShardLevels& L, int world, int workers_per_rank1,
                       int workers_per_rank2, Split* sp1, Split* sp2) {
    const int64_t ld = round_up(n, 256);
    plan_split(sp1, n, NT * P1_R, L.sym ? 0 : W_ALL[L.level1], W_HEAD[L.level1], 0, world * workers_per_rank1, ld, 12,
               (size_t)-1);
    plan_split(sp2, n, NT * P2_R, W2_PLAIN, W2_OWN, 1, world * workers_per_rank2, ld, 2, (size_t)-1);
    (void)ctx;
}

// Partial slots of the sharded cut.  With world x W workers on the axis a tile may be shared by up to min(its workers, W)
// workers of one rank -- world times what the one-GPU cut needs -- so the sharded phases keep partial buffers of their
// own, sized for the cut at hand and grown on demand (the one allocation of these calls; kept by the context).
inline int shard_slots_bound(const Split& sp, int workers_per_rank) {
    int worst = 0;
    for (int I = 0; I < sp.n_tiles; ++I) {
        int first, count;
        split_slots(sp, I, &first, &count);            // sp.w_begin / w_end still span the whole axis here
        if (count > workers_per_rank) count = workers_per_rank;
        if (count > worst) worst = count;
    }
    return worst;
}
inline int shard_ensure(double** buf, size_t* have, size_t need) {
    if (need <= *have) return HAWKES_OK;
    if (*buf) cudaFree(*buf);
    *buf = nullptr;
    *have = 0;
    if (cudaMalloc((void**)buf, need * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return HAWKES_ERR_NOMEM; }
    *have = need;
    return HAWKES_OK;
}

template <bool DIM3>
int shard_pass1_impl(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta, const DevConsts& c,
                     const ShardLevels& L, int rank, int world, double* part_out, cudaStream_t st) {
    const int W1 = ctx->sm_count * ctx->occ1[L.level1], W2 = ctx->sm_count * ctx->occ2[L.level2];
    Split sp1, sp2;
    shard_plan(ctx, n, L, world, W1, W2, &sp1, &sp2);
    const int64_t ld = round_up(n, 256);
    {
        const int rc = shard_ensure(&ctx->d_shpart1, &ctx->shpart1_doubles, (size_t)shard_slots_bound(sp1, W1) * 12 * (size_t)ld);
        if (rc) return rc;
    }
    sp1.w_begin = rank * W1;
    sp1.w_end = (rank + 1) * W1;
    const int nblk = (int)((n + RED_T - 1) / RED_T);
    CK(cudaMemsetAsync(ctx->d_status, 0, 2 * sizeof(unsigned), st));
    prep_kernel<<<nblk, RED_T, 0, st>>>(n, ctx->dim, x, t, theta, ctx->d_rec, ctx->d_status, c.omega);
    const unsigned g1 = (unsigned)ctx->sm_count;
    const int lv = L.level1;
#define SHARD_P1(LV)                                                                                                        \
    if (L.sym)                                                                                                              \
        pass1s_kernel<P1_R, (LV) <= 1 ? (LV) : 1, DIM3, P1_G[(LV) <= 1 ? (LV) : 1]>                                         \
            <<<g1, NT * P1_G[LV], smem_request(P1_G[LV] * sym_group_bytes<DIM3>((LV) == 0 ? 1 : 3)), st>>>(                 \
                ctx->d_rec, n, ld, c, ctx->d_tab, ctx->d_shpart1, ctx->d_partc, sp1);                                         \
    else                                                                                                                    \
        pass1_kernel<P1_R, LV, DIM3, P1_G[LV]><<<g1, NT * P1_G[LV], smem_request(P1_G[LV] * group_buf_bytes<DIM3>()), st>>>( \
            ctx->d_rec, n, ld, c, ctx->d_tab, ctx->d_shpart1, sp1);                                                           \
    shard_sum1_kernel<LV><<<nblk, RED_T, 0, st>>>(n, ld, ctx->d_shpart1, sp1, L.sym ? ctx->d_partc : nullptr, NT * P1_R, part_out)
    if (lv == 0) { SHARD_P1(0); }
    else if (lv == 1) { SHARD_P1(1); }
    else { SHARD_P1(2); }
#undef SHARD_P1
    ctx->launches += 3;
    CK(cudaGetLastError());
    return HAWKES_OK;
}

template <bool DIM3>
int shard_reduce1_impl(hawkes_ctx* ctx, int64_t n, const DevConsts& c, uint32_t want, const ShardLevels& L, int world,
                       const double* parts_all, double* ll, double* grad_hyper, double* hess_hyper, cudaStream_t st) {
    const int64_t ld = round_up(n, 256);
    const int nblk = (int)((n + RED_T - 1) / RED_T);
    Split sg{};                    // the gathered sums: `world` slots per tile, [rank][moment][ld]
    sg.n = n;
    sg.tile = NT * P1_R;
    sg.n_tiles = (int)((n + sg.tile - 1) / sg.tile);
    sg.chunk = 1;
    sg.fixed_slots = world;
    double* const rowd1 = L.level1 >= 1 ? ctx->d_rowd1 : nullptr;
    double* const rowd2 = L.level1 >= 2 ? ctx->d_rowd2 : nullptr;
#define SHARD_R1(LV)                                                                                                        \
    reduce1_kernel<LV, DIM3><<<nblk, RED_T, 0, st>>>(ctx->d_rec, n, ld, c, parts_all, sg, ctx->d_lam, ctx->d_trec,          \
                                                     ctx->d_trec2, rowd1, rowd2, nullptr, ctx->d_blockpart, ctx->d_status,  \
                                                     ctx->d_bgcache, 0, nullptr, sg.n_tiles, NT * P1_R, nullptr)
    if (L.level1 == 0) { SHARD_R1(0); }
    else if (L.level1 == 1) { SHARD_R1(1); }
    else { SHARD_R1(2); }
#undef SHARD_R1
    ctx->launches++;
    if (want & (HAWKES_WANT_LL | HAWKES_WANT_GRAD_HYPER | HAWKES_WANT_HESS_HYPER)) {
        scalars_kernel<<<1, SCAL_T, 0, st>>>(ctx->d_blockpart, nblk, c, (want & HAWKES_WANT_LL) ? ll : nullptr,
                                             (want & HAWKES_WANT_GRAD_HYPER) ? grad_hyper : nullptr,
                                             (want & HAWKES_WANT_HESS_HYPER) ? hess_hyper : nullptr, ctx->d_scal);
        ctx->launches++;
    }
    CK(cudaGetLastError());
    return HAWKES_OK;
}

template <bool DIM3>
int shard_pass2_impl(hawkes_ctx* ctx, int64_t n, const DevConsts& c, const ShardLevels& L, int rank, int world,
                     double* part2_out, cudaStream_t st) {
    const int W1 = ctx->sm_count * ctx->occ1[L.level1], W2 = ctx->sm_count * ctx->occ2[L.level2];
    Split sp1, sp2;
    shard_plan(ctx, n, L, world, W1, W2, &sp1, &sp2);
    const int64_t ld = round_up(n, 256);
    {
        const int rc = shard_ensure(&ctx->d_shpart2, &ctx->shpart2_doubles, (size_t)shard_slots_bound(sp2, W2) * 2 * (size_t)ld);
        if (rc) return rc;
    }
    sp2.w_begin = rank * W2;
    sp2.w_end = (rank + 1) * W2;
    const int nblk = (int)((n + RED_T - 1) / RED_T);
    const unsigned g2 = (unsigned)ctx->sm_count;
    if (L.level2)
        pass2_kernel<P2_R, 1, DIM3, P2_G[1]><<<g2, NT * P2_G[1], smem_request(P2_G[1] * group_buf_bytes<DIM3>()), st>>>(
            ctx->d_rec, ctx->d_trec, ctx->d_trec2, ctx->d_status, n, ld, c, ctx->d_tab, ctx->d_shpart2, sp2);
    else
        pass2_kernel<P2_R, 0, DIM3, P2_G[0]><<<g2, NT * P2_G[0], smem_request(P2_G[0] * group_buf_bytes<DIM3>()), st>>>(
            ctx->d_rec, ctx->d_trec, ctx->d_trec2, ctx->d_status, n, ld, c, ctx->d_tab, ctx->d_shpart2, sp2);
    shard_sum2_kernel<<<nblk, RED_T, 0, st>>>(n, ld, ctx->d_shpart2, sp2, L.level2, part2_out);
    ctx->launches += 2;
    CK(cudaGetLastError());
    return HAWKES_OK;
}

template <bool DIM3>
int shard_finish_impl(hawkes_ctx* ctx, int64_t n, const DevConsts& c, uint32_t want, int world, const double* parts2_all,
                      double* grad_theta, double* hess_theta_diag, cudaStream_t st) {
    const int64_t ld = round_up(n, 256);
    const int nblk = (int)((n + RED_T - 1) / RED_T);
    Split sg{};
    sg.n = n;
    sg.tile = NT * P2_R;
    sg.n_tiles = (int)((n + sg.tile - 1) / sg.tile);
    sg.chunk = 1;
    sg.fixed_slots = world;
    theta_kernel<DIM3><<<nblk, RED_T, 0, st>>>(ctx->d_rec, n, ld, c, parts2_all, sg,
                                               (want & HAWKES_WANT_GRAD_THETA) ? grad_theta : nullptr,
                                               (want & HAWKES_WANT_HESS_THETA) ? hess_theta_diag : nullptr, nullptr, nullptr);
    ctx->launches++;
    CK(cudaGetLastError());
    return HAWKES_OK;
}
