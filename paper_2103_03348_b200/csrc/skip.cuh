// Exact-zero skipping: a variant of the pairwise passes that visits only those tile
// pairs which can hold a non-zero term of Eq. 1 / Eq. 4, reported separately from the
// dense path (the paper's method visits every pair).
//
// A term exp(-z) of either kernel is exactly +0.0 in IEEE double arithmetic once z > 1075 ln 2 = 745.14.  The
// events are re-ordered as the leaves of a space-time k-d tree (median splits along the axis of furthest reach in
// units of the cut-off radius; leaves = the runs of TS records the kernels stream), every run gets a bounding
// box in space and time, and a (target tile, source chunk) pair is dropped when the smallest exponent any of
// its pairs can have exceeds SKIP_Z0 = 746 -- or, for the excitation term, when no pair of it is causal.  Only
// exact zeros are dropped: every sum changes by its summation order alone.  In the tree order time is no
// longer sorted, so every excitation pair takes the per-pair test dt > 0 (MODE 2 / MASKED of the dense tiles).
//
// The plan (order, boxes, work lists, their cut into workers) is built on the host by hawkes_skip_plan: it
// depends on the events and the hyperparameters, not on theta, so one plan serves every evaluation of an HMC
// trajectory.  Included by hawkes.cu after its kernels and the context struct.
#include <algorithm>
#include <cstring>
#include <vector>

namespace {

constexpr double SKIP_Z0 = 746.0;      // exp(-z) == +0.0 for z >= 745.14
constexpr int SK_B = 1, SK_S = 2;      // item kinds: background live, excitation live (3 = both)
static_assert(P1_G[0] == P1_G[1] && P1_G[1] == P1_G[2] && P2_G[0] == P2_G[1], "one worker count per pass");

// a0': pack the caller's event perm[i] into record i; times need not be sorted here.
__global__ void skip_gather_kernel(int64_t n, int dim, const int64_t* __restrict__ perm, const double* __restrict__ x,
                                   const double* __restrict__ t, const double* __restrict__ theta,
                                   double* __restrict__ rec, unsigned* __restrict__ status) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t o = perm[i];
    const double ti = t[o], th = theta[o];
    unsigned bad = 0;
    if (!isfinite(ti) || !isfinite(th) || th < 0.0) bad |= ST_NONFINITE;
    double xv[3] = {0.0, 0.0, 0.0};
    for (int d = 0; d < dim; ++d) {
        xv[d] = x[(int64_t)d * n + o];
        if (!isfinite(xv[d])) bad |= ST_NONFINITE;
    }
    if (dim <= 2) {
        reinterpret_cast<double4*>(rec)[i] = make_double4(xv[0], xv[1], ti, th);
    } else {
        double2* r2 = reinterpret_cast<double2*>(rec) + 3 * i;
        r2[0] = make_double2(xv[0], xv[1]);
        r2[1] = make_double2(xv[2], ti);
        r2[2] = make_double2(th, 0.0);
    }
    if (bad) atomicOr(status, bad);
}

// a1 over a work list.  items[k] = (target tile I of NT*R records, source chunk J of TS records * 4 + kind), sorted
// by I then J; worker w (one group of NT threads) takes items [wstart[w], wstart[w+1]) and writes, for every tile
// it touches, partial slot (w - wfirst[I]) in the layout of pass1_kernel.
template <int R, int LEVEL, bool DIM3, int G>
__global__ void __launch_bounds__(NT * G, 1) pass1_list_kernel(const double* __restrict__ rec, int64_t n, int64_t ld,
                                                               DevConsts c, const double* __restrict__ tab_g,
                                                               double* __restrict__ part, const int2* __restrict__ items,
                                                               const int* __restrict__ wstart,
                                                               const int* __restrict__ wfirst, int n_workers) {
    constexpr int RS = DIM3 ? 6 : 4;
    constexpr int NB = Mom<LEVEL>::NB;
    constexpr unsigned BUF = group_buf_bytes<DIM3>();
    static_assert(smem_request(G * BUF) <= SMEM_MAX, "table + streaming buffers must fit shared memory");
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double smagic;
    const unsigned smem_base = (unsigned)__cvta_generic_to_shared(smem);
    const SmemPlan plan = smem_plan(smem_base, G * BUF);
    fill_table(reinterpret_cast<double*>(smem + plan.tab_off), tab_g);
    stash_consts(smagic);
    __syncthreads();

    const int grp = threadIdx.x / NT, tid = threadIdx.x % NT;
    const int w = blockIdx.x * G + grp;
    if (w >= n_workers) return;
    const int q0 = wstart[w], q1 = wstart[w + 1];   // in 32-record blocks, 4 per item
    if (q0 >= q1) return;
    const int k0 = q0 / 4, k1 = (q1 - 1) / 4 + 1;
    double* const sbuf0 = reinterpret_cast<double*>(smem + plan.buf_off + grp * BUF);
    double* const sbuf1 = sbuf0 + TS * RS;
    const unsigned lane_base = (smem_base + plan.tab_off) | (8u * (threadIdx.x & 31));
    const P1C pc = pinned_consts(smagic, c);

    // the piece of item k this worker holds: streamed records [a, a + cnt)
    auto piece = [&](int k, int y, int64_t* a, int* cnt) {
        const int jb = k == q0 / 4 ? q0 % 4 : 0;
        const int je = k == (q1 - 1) / 4 ? (q1 - 1) % 4 + 1 : 4;
        const int64_t c0 = (int64_t)(y >> 2) * TS;
        *a = c0 + jb * 32;
        *cnt = (int)max(min(c0 + je * 32, n) - *a, (int64_t)0);
    };
    Ev<DIM3> g[R];
    Mom<LEVEL> m[R];
    auto flush = [&](int I) {
        const int slot = w - wfirst[I];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = (int64_t)I * (NT * R) + r * NT + tid;
            if (i < n) {
                double* o = part + (int64_t)slot * (2 * NB) * ld + i;
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    o[(int64_t)k * ld] = m[r].b[k];
                    o[(int64_t)(NB + k) * ld] = m[r].s[k];
                }
            }
        }
    };

    RecIO<DIM3> io;
    int2 it = items[k0];
    int64_t a, a2 = 0;
    int cnt, cnt2 = 0;
    piece(k0, it.y, &a, &cnt);
    io.load(rec, a, cnt, tid);
    io.store(sbuf0, tid);
    group_sync(grp);
    int cur = 0, I = -1;
    for (int k = k0; k < k1; ++k) {
        if (it.x != I) {
            if (I >= 0) flush(I);
            I = it.x;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int64_t i = min((int64_t)I * (NT * R) + r * NT + tid, n - 1);
                g[r] = read_rec<DIM3>(rec + i * RS);
#pragma unroll
                for (int q = 0; q < NB; ++q) { m[r].b[q] = 0.0; m[r].s[q] = 0.0; }
            }
        }
        int2 nx = it;
        if (k + 1 < k1) {
            nx = items[k + 1];
            piece(k + 1, nx.y, &a2, &cnt2);
            io.load(rec, a2, cnt2, tid);
        }
        const double* sb = cur ? sbuf1 : sbuf0;
        const int kind = it.y & 3;
        if (kind == SK_B) p1_tile<R, LEVEL, 0, DIM3, true>(sb, cnt, g, m, pc, lane_base);
        else if (kind == SK_S) p1_tile<R, LEVEL, 2, DIM3, false>(sb, cnt, g, m, pc, lane_base);
        else p1_tile<R, LEVEL, 2, DIM3, true>(sb, cnt, g, m, pc, lane_base);
        if (k + 1 < k1) io.store(cur ? sbuf0 : sbuf1, tid);
        group_sync(grp);
        cur ^= 1;
        it = nx;
        a = a2;
        cnt = cnt2;
    }
    flush(I);
}

// a4 over a work list: items[k] = (source tile M of NT*R records, target chunk J * 4 + SK_S); the targets
// (x, t, 1/lambda) stream from trec and every pair takes the test t_n > t_m.
template <int R, int LEVEL, bool DIM3, int G>
__global__ void __launch_bounds__(NT * G, 1) pass2_list_kernel(const double* __restrict__ rec, const double* __restrict__ trec,
                                                               int64_t n, int64_t ld, DevConsts c,
                                                               const double* __restrict__ tab_g, double* __restrict__ part2,
                                                               const int2* __restrict__ items, const int* __restrict__ wstart,
                                                               const int* __restrict__ wfirst, int n_workers) {
    constexpr int RS = DIM3 ? 6 : 4;
    constexpr unsigned BUF = group_buf_bytes<DIM3>();
    static_assert(smem_request(G * BUF) <= SMEM_MAX, "table + streaming buffers must fit shared memory");
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double smagic;
    const unsigned smem_base = (unsigned)__cvta_generic_to_shared(smem);
    const SmemPlan plan = smem_plan(smem_base, G * BUF);
    fill_table(reinterpret_cast<double*>(smem + plan.tab_off), tab_g);
    stash_consts(smagic);
    __syncthreads();

    const int grp = threadIdx.x / NT, tid = threadIdx.x % NT;
    const int w = blockIdx.x * G + grp;
    if (w >= n_workers) return;
    const int q0 = wstart[w], q1 = wstart[w + 1];   // in 32-record blocks, 4 per item
    if (q0 >= q1) return;
    const int k0 = q0 / 4, k1 = (q1 - 1) / 4 + 1;
    double* const sbuf0 = reinterpret_cast<double*>(smem + plan.buf_off + grp * BUF);
    double* const sbuf1 = sbuf0 + TS * RS;
    const unsigned lane_base = (smem_base + plan.tab_off) | (8u * (threadIdx.x & 31));
    const P1C pc = pinned_consts(smagic, c);

    auto piece = [&](int k, int y, int64_t* a, int* cnt) {
        const int jb = k == q0 / 4 ? q0 % 4 : 0;
        const int je = k == (q1 - 1) / 4 ? (q1 - 1) % 4 + 1 : 4;
        const int64_t c0 = (int64_t)(y >> 2) * TS;
        *a = c0 + jb * 32;
        *cnt = (int)max(min(c0 + je * 32, n) - *a, (int64_t)0);
    };
    Ev<DIM3> g[R];
    double cm[R], dm[R];
    auto flush = [&](int M) {
        const int slot = w - wfirst[M];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = (int64_t)M * (NT * R) + r * NT + tid;
            if (i < n) {
                part2[(int64_t)(slot * 2 + 0) * ld + i] = cm[r];
                if (LEVEL >= 1) part2[(int64_t)(slot * 2 + 1) * ld + i] = dm[r];
            }
        }
    };

    RecIO<DIM3> io;
    int2 it = items[k0];
    int64_t a, a2 = 0;
    int cnt, cnt2 = 0;
    piece(k0, it.y, &a, &cnt);
    io.load(trec, a, cnt, tid);
    io.store(sbuf0, tid);
    group_sync(grp);
    int cur = 0, M = -1;
    for (int k = k0; k < k1; ++k) {
        if (it.x != M) {
            if (M >= 0) flush(M);
            M = it.x;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int64_t i = min((int64_t)M * (NT * R) + r * NT + tid, n - 1);
                g[r] = read_rec<DIM3>(rec + i * RS);
                cm[r] = 0.0;
                dm[r] = 0.0;
            }
        }
        int2 nx = it;
        if (k + 1 < k1) {
            nx = items[k + 1];
            piece(k + 1, nx.y, &a2, &cnt2);
            io.load(trec, a2, cnt2, tid);
        }
        p2_tile<R, LEVEL, true, DIM3>(cur ? sbuf1 : sbuf0, cnt, g, cm, dm, pc, lane_base);
        if (k + 1 < k1) io.store(cur ? sbuf0 : sbuf1, tid);
        group_sync(grp);
        cur ^= 1;
        it = nx;
        a = a2;
        cnt = cnt2;
    }
    flush(M);
}


// a1, background term over a list, once per UNORDERED pair (pass1_sym.cuh: row sums in registers, column sums in an
// accumulator that rotates through the warp).  items[k] = (target tile I, source chunk J) with J <= the last chunk of
// tile I: the pairs (target i of I, source j of J, j < i).  Work is cut in units of 32-source blocks (4 per item):
// worker w takes the blocks [wstart[w], wstart[w+1]) of the flattened (item, block) sequence; a column partial
// (tile I, source j) is written by the one worker that holds j's block, a row partial slot per worker as elsewhere.
// The excitation sums of the slot are written as zeros (the S items have their own slots, after these).
template <int R, int LEVEL, bool DIM3, int G>
__global__ void __launch_bounds__(NT * G, 1) pass1_symb_list_kernel(const double* __restrict__ rec, int64_t n, int64_t ld,
                                                                    DevConsts c, const double* __restrict__ tab_g,
                                                                    double* __restrict__ part, double* __restrict__ partc,
                                                                    int n_tiles, const int2* __restrict__ items,
                                                                    const int* __restrict__ wstart,
                                                                    const int* __restrict__ wfirst, int n_workers) {
    constexpr int RS = DIM3 ? 6 : 4;
    constexpr int NB = Mom<LEVEL>::NB;
    constexpr int NA = SoaIO<DIM3>::NA;
    constexpr unsigned GB = sym_group_bytes<DIM3>(NB);
    static_assert(smem_request(G * GB) <= SMEM_MAX, "table + group buffers must fit shared memory");
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ P1C spc;
    const unsigned smem_base = (unsigned)__cvta_generic_to_shared(smem);
    const SmemPlan plan = smem_plan(smem_base, G * GB);
    fill_table(reinterpret_cast<double*>(smem + plan.tab_off), tab_g);
    if (threadIdx.x == 0)
        spc = P1C{c.negcb, c.negcs, c.rho_b, c.rho_s, c.lim_b_hi, c.lim_s_hi, {c.d0, c.d1, c.d2, c.d3, MAGIC}};
    __syncthreads();

    const int grp = threadIdx.x / NT, tid = threadIdx.x % NT, lane = threadIdx.x & 31, wrp = tid >> 5;
    const int w = blockIdx.x * G + grp;
    if (w >= n_workers) return;
    const int q0 = wstart[w], q1 = wstart[w + 1];
    if (q0 >= q1) return;
    double* const gbuf = reinterpret_cast<double*>(smem + plan.buf_off + grp * GB);
    double* const sbuf0 = gbuf;
    double* const sbuf1 = gbuf + NA * TS;
    double* const colacc = gbuf + 2 * NA * TS;            // [NT/32][TS][NB]
    double* const mycol = colacc + wrp * TS * NB;
    const unsigned lane_base = (smem_base + plan.tab_off) | (8u * lane);
    P1C pc;
    {
        const volatile P1C& v = spc;
        pc.negcb = v.negcb; pc.negcs = v.negcs; pc.rho_b = v.rho_b; pc.rho_s = v.rho_s;
        pc.lim_b_hi = v.lim_b_hi; pc.lim_s_hi = v.lim_s_hi;
        pc.e.d0 = v.e.d0; pc.e.d1 = v.e.d1; pc.e.d2 = v.e.d2; pc.e.d3 = v.e.d3; pc.e.magic = v.e.magic;
    }

    Ev<DIM3> g[R];
    int64_t gi[R];
    Mom<LEVEL> m[R];
    auto flush = [&](int I) {
        const int slot = w - wfirst[I];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = (int64_t)I * (NT * R) + r * NT + tid;
            if (i < n) {
                double* o = part + (int64_t)slot * (2 * NB) * ld + i;
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    o[(int64_t)k * ld] = m[r].b[k];
                    o[(int64_t)(NB + k) * ld] = 0.0;
                }
            }
        }
    };
    // the piece of item k this worker holds: source records [a, a + cnt)
    auto piece = [&](int k, int64_t* a, int* cnt) {
        const int jb = k == q0 / 4 ? q0 % 4 : 0;
        const int je = k == (q1 - 1) / 4 ? (q1 - 1) % 4 + 1 : 4;
        const int64_t c0 = (int64_t)items[k].y * TS;
        *a = c0 + jb * 32;
        const int64_t e = min(c0 + je * 32, n);
        *cnt = (int)max(e - *a, (int64_t)0);
    };

    SoaIO<DIM3> io;
    const int k_first = q0 / 4, k_last = (q1 - 1) / 4;
    int64_t a, a2 = 0;
    int cnt, cnt2 = 0;
    piece(k_first, &a, &cnt);
    io.load(rec, a, cnt, tid);
    io.store(sbuf0, tid);
    group_sync(grp);
    int cur = 0, I = -1;
    bool ragged_tile = false;
    for (int k = k_first; k <= k_last; ++k) {
        const int It = items[k].x;
        if (It != I) {
            if (I >= 0) flush(I);
            I = It;
            const int64_t i0 = (int64_t)I * (NT * R);
            ragged_tile = n - i0 < NT * R;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int64_t i = i0 + r * NT + tid;
                gi[r] = i < n ? i : -1;
                g[r] = read_rec<DIM3>(rec + min(i, n - 1) * RS);
#pragma unroll
                for (int q = 0; q < NB; ++q) { m[r].b[q] = 0.0; m[r].s[q] = 0.0; }
            }
        }
        if (k < k_last) {
            piece(k + 1, &a2, &cnt2);
            io.load(rec, a2, cnt2, tid);
        }
        const double* sb = cur ? sbuf1 : sbuf0;
        const bool plain = !ragged_tile && a + cnt <= (int64_t)I * (NT * R);   // every source index below every target's
        for (int j0 = 0; j0 < cnt; j0 += 32) {
            const int nvalid = min(32, cnt - j0);
            if (plain && nvalid == 32)
                p1s_block<R, LEVEL, false, DIM3, false>(sb, j0, nvalid, a + j0, g, gi, m, mycol, pc, lane_base, lane);
            else
                p1s_block<R, LEVEL, true, DIM3, false>(sb, j0, nvalid, a + j0, g, gi, m, mycol, pc, lane_base, lane);
        }
        if (k < k_last) io.store(cur ? sbuf0 : sbuf1, tid);
        group_sync(grp);
        if (tid < cnt) {   // column sums of this piece: the four warps' shares in warp order, one source per thread
            const int64_t j = a + tid;
            const int sl = I - (int)(j / (NT * R));
#pragma unroll
            for (int q = 0; q < NB; ++q) {
                double v = 0.0;
#pragma unroll
                for (int ww = 0; ww < NT / 32; ++ww) v += colacc[(ww * TS + tid) * NB + q];
                partc[colpart_index(n_tiles, NT * R, NB, sl, q, j)] = v;
            }
        }
        group_sync(grp);
        cur ^= 1;
        a = a2;
        cnt = cnt2;
    }
    flush(I);
}

}  // namespace

// -------------------------------------------------------------------------------------------------
// host side: the plan
struct SkipPlan {
    int64_t n;
    hawkes_params p;
    int s_mode;
    int64_t* d_perm;       // record i of the tree order is the caller's event perm[i]
    int2* d_pool_items;    // one allocation for the four item lists (the d_items* pointers point into it)
    int* d_pool_cut;       // ... and one for their cuts (d_w*start, d_w*first, d_slots*, ...)
    double* d_ev;          // the planned events as the caller gave them (x, then t): a re-plan recognises them on the device
    double* d_tn;          // t_N = max t
    int2* d_items1;        // pass-1 work list and its cut
    int* d_w1start;
    int* d_w1first;
    int* d_slots1;
    int workers1;
    int2* d_items1s;       // pass 1 without the background term (cached sums, hawkes_hmc_run): the S items alone
    int* d_w1sstart;
    int* d_w1sfirst;
    int* d_slots1s;
    int workers1s;
    // symmetric background (levels 0 and 1): unordered (tile, chunk) items cut in 32-source blocks, the S items after
    // them in every tile's slots, and the plan's own column partials (zero wherever no item writes)
    int2* d_itemsb;
    int* d_wbstart;
    int* d_wbfirst;
    int* d_w1sfirst_sym;
    int* d_slots_sym;
    int workersb;
    double* d_partc;
    size_t partc_doubles;
    size_t part_sym_doubles;
    double* d_part_sym;    // row partials of that form: the late tiles of the unordered enumeration take more slots
                           // than the context's buffer is sized for
    int partc_level;       // NB layout the buffer currently holds (-1: freshly zeroed)
    int64_t items_bsym;
    int2* d_items2;        // pass-2 work list and its cut
    int* d_w2start;
    int* d_w2first;
    int* d_slots2;
    int workers2;
    // what the lists hold, for hawkes_skip_stats
    int64_t items_b, items_s, items_p2, items_dense1, items_dense2;
    // host copy of the planned events, their order and boxes: a re-plan for other hyperparameters of the same events
    // (an MCMC sweep changes them between HMC updates) keeps the order while the cut-off radii stay within a factor 2
    // of those it was built for -- any order is valid, the boxes are exact for it -- and only rebuilds the lists
    struct SkipHost* host;
    int order_reused;
};

namespace {

// One SM is left free: hawkes_posterior_z_skip runs the single-CTA tree prior on the side stream beside the list
// kernels, and a CTA of theirs that had to wait for that SM would hold up the whole pass.
inline int skip_sms(const hawkes_ctx* ctx) { return ctx->sm_count > 1 ? ctx->sm_count - 1 : 1; }

struct SkipBox {           // bounding box of a run of records: up to 3 coordinates, then time
    double lo[4], hi[4];
};
}  // namespace
struct SkipHost {
    std::vector<double> hx, ht;
    std::vector<int64_t> perm;
    std::vector<SkipBox> chunk, tile;
    double cutoff[4];
};
namespace {

void skip_plan_free(hawkes_ctx* c) {
    SkipPlan* s = c->skip;
    if (!s) return;
    void* ptrs[] = {s->d_ev, s->d_perm, s->d_tn, s->d_pool_items, s->d_pool_cut, s->d_partc, s->d_part_sym};
    for (void* q : ptrs)
        if (q) cudaFree(q);
    delete s->host;
    delete s;
    c->skip = nullptr;
}


// The box tests, one definition for the host and the device.  (targets T, sources S)
struct SkipGeom {
    int dim, s_mode;
    double tau_x, tau_t, h, omega;
};
__host__ __device__ inline double skip_gap2(const SkipBox& A, const SkipBox& B, int dim) {   // squared distance of the spatial boxes
    double s = 0.0;
    for (int a = 0; a < dim; ++a) {
        const double g = fmax(0.0, fmax(A.lo[a] - B.hi[a], B.lo[a] - A.hi[a]));
        s += g * g;
    }
    return s;
}
// background: smallest exponent r^2/2tau_x^2 + dt^2/2tau_t^2 any pair of the boxes can have
__host__ __device__ inline bool skip_live_b(const SkipBox& T, const SkipBox& S, const SkipGeom& q) {
    double z = skip_gap2(T, S, q.dim) / (2.0 * q.tau_x * q.tau_x);
    if (!q.s_mode) {
        const double g = fmax(0.0, fmax(T.lo[q.dim] - S.hi[q.dim], S.lo[q.dim] - T.hi[q.dim]));
        z += g * g / (2.0 * q.tau_t * q.tau_t);
    }
    return !(z >= SKIP_Z0);
}
// excitation of targets T by sources S: some pair must be causal (t_n > t_m); smallest exponent r^2/2h^2 + omega dt
__host__ __device__ inline bool skip_live_s(const SkipBox& T, const SkipBox& S, const SkipGeom& q) {
    if (!(T.hi[q.dim] > S.lo[q.dim])) return false;
    const double z = skip_gap2(T, S, q.dim) / (2.0 * q.h * q.h) + q.omega * fmax(0.0, T.lo[q.dim] - S.hi[q.dim]);
    return !(z >= SKIP_Z0);
}

// The four work lists on the device: one thread per (tile I, tile Jt) pair tests the tile boxes, then the CPT chunks of
// Jt against tile I.  Pass A counts (cnt[l][I*nt + Jt], l = 0: pass-1 items of either kind, 1: with a live excitation,
// 2: unordered background items (Jt <= I), 3: pass-2 items of source tile I and target tile Jt); an exclusive scan of
// each count array gives the offsets; pass B (FILL) writes the items there -- sorted by I, then J, as the host loops
// of round 1 produced them.
constexpr int SKIP_CPT = (NT * P1_R) / TS;   // chunks per tile
template <bool FILL>
__global__ void __launch_bounds__(256) skip_lists_kernel(int nt, int nc, const SkipBox* __restrict__ tile,
                                                         const SkipBox* __restrict__ chunk, SkipGeom q,
                                                         int* __restrict__ cnt, const int* __restrict__ off,
                                                         int2* __restrict__ items1, int2* __restrict__ items1s,
                                                         int2* __restrict__ itemsb, int2* __restrict__ items2) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t np = (int64_t)nt * nt;
    if (idx >= np) return;
    const int I = (int)(idx / nt), Jt = (int)(idx % nt);
    const SkipBox TI = tile[I], TJ = tile[Jt];
    const bool tb = skip_live_b(TI, TJ, q), ts = skip_live_s(TI, TJ, q), t2 = skip_live_s(TJ, TI, q);
    int c1 = 0, c1s = 0, cb = 0, c2 = 0;
    int o1 = 0, o1s = 0, ob = 0, o2 = 0;
    if (FILL) { o1 = off[idx]; o1s = off[np + idx]; ob = off[2 * np + idx]; o2 = off[3 * np + idx]; }
    if (tb || ts || t2) {
        for (int J = Jt * SKIP_CPT; J < min(nc, (Jt + 1) * SKIP_CPT); ++J) {
            const SkipBox C = chunk[J];
            const bool lb = tb && skip_live_b(TI, C, q), ls = ts && skip_live_s(TI, C, q);
            const int kind = (lb ? SK_B : 0) | (ls ? SK_S : 0);
            if (kind) {
                if (FILL) items1[o1 + c1] = make_int2(I, J * 4 + kind);
                ++c1;
            }
            if (ls) {
                if (FILL) items1s[o1s + c1s] = make_int2(I, J * 4 + SK_S);
                ++c1s;
            }
            if (lb && Jt <= I) {
                if (FILL) itemsb[ob + cb] = make_int2(I, J);
                ++cb;
            }
            if (t2 && skip_live_s(C, TI, q)) {      // pass 2: sources = tile I, targets = chunk J
                if (FILL) items2[o2 + c2] = make_int2(I, J * 4 + SK_S);
                ++c2;
            }
        }
    }
    if (!FILL) { cnt[idx] = c1; cnt[np + idx] = c1s; cnt[2 * np + idx] = cb; cnt[3 * np + idx] = c2; }
}

// Device-side cut of a work list (sorted by tile) into `workers` consecutive ranges of about equal cost, in units of
// 32-record blocks (4 per item; cost[k] = cost of one block of item k, NULL: 1; C = exclusive prefix sum of cost, NULL: k).
// wstart[w], w = 0..workers: first block of worker w (workers at the end of a short list may be empty); tile_start[I],
// I = 0..n_tiles: first item of tile I.  The same cut whatever the launch: it depends on the list alone.
__device__ __forceinline__ long long skip_before(const long long* C, int k) { return C ? 4 * C[k] : 4ll * k; }
__global__ void skip_cut_kernel(const int2* __restrict__ items, int K, const int* __restrict__ cost,
                                const long long* __restrict__ C, int workers, int n_tiles, int* __restrict__ wstart,
                                int* __restrict__ tile_start) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = K > 0 ? skip_before(C, K - 1) + 4ll * (cost ? cost[K - 1] : 1) : 0;
    const long long chunk = (total + workers - 1) / workers > 0 ? (total + workers - 1) / workers : 1;
    if (i <= workers) {
        int v;
        const long long T = (long long)i * chunk;          // worker i starts once the cost before it reaches T
        if (i == 0 || K == 0) v = 0;
        else if (T >= total) v = 4 * K;
        else {
            int lo = 0, hi = K - 1;                          // largest k with skip_before(k) < T
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (skip_before(C, mid) < T) lo = mid; else hi = mid - 1;
            }
            const long long ck = cost ? cost[lo] : 1;
            long long b = (T - skip_before(C, lo) + ck - 1) / ck - 1;   // block of item lo at whose end T is reached
            if (b < 0) b = 0;
            if (b > 3) b = 3;
            v = 4 * lo + (int)b + 1;
            if (v > 4 * K) v = 4 * K;
        }
        if (i == workers) v = 4 * K;
        wstart[i] = v;
    }
    if (i <= n_tiles) {
        int lo = 0, hi = K;                                  // first item with tile >= i
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (items[mid].x < i) lo = mid + 1; else hi = mid;
        }
        tile_start[i] = lo;
    }
}
// Workers that came out empty (two thresholds inside one block of a short list) move to the end: every tile's workers
// are then consecutive and non-empty, as the partial-slot numbering (worker - first worker of the tile) assumes.
__global__ void skip_compact_kernel(int workers, int nblocks, int* __restrict__ wstart) {
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    int used = 0;                                            // wstart[0..used] strictly increasing so far
    for (int w = 1; w <= workers; ++w)
        if (wstart[w] > wstart[used]) wstart[++used] = wstart[w];
    for (int w = used + 1; w <= workers; ++w) wstart[w] = nblocks;
}
// per tile: the first worker that holds one of its blocks and the number of workers that do (= partial slots)
__global__ void skip_slots_kernel(int n_tiles, int workers, const int* __restrict__ wstart, const int* __restrict__ tile_start,
                                  int* __restrict__ wfirst, int* __restrict__ slots, int* __restrict__ worst) {
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_tiles) return;
    const int k0 = tile_start[I], k1 = tile_start[I + 1];
    int first = 0, count = 0;
    if (k1 > k0) {
        auto worker_of = [&](int q) {                        // the worker w with wstart[w] <= q < wstart[w + 1]
            int lo = 0, hi = workers - 1;
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (wstart[mid] <= q) lo = mid; else hi = mid - 1;
            }
            return lo;
        };
        first = worker_of(4 * k0);
        count = worker_of(4 * k1 - 1) - first + 1;
    }
    wfirst[I] = first;
    slots[I] = count;
    atomicMax(worst, count);
}
__global__ void skip_cost1_kernel(int K, const int2* __restrict__ items, int wb, int ws, int* __restrict__ cost,
                                  unsigned long long* __restrict__ n_b) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const int kind = items[k].y & 3;
    cost[k] = ((kind & SK_B) ? wb : 0) + ((kind & SK_S) ? ws : 0);
    if (kind & SK_B) atomicAdd(n_b, 1ull);
}
// symmetric form: the S items' slots follow the unordered background items' in every tile
__global__ void skip_sym_kernel(int n_tiles, const int* __restrict__ wf_s, const int* __restrict__ sl_s,
                                const int* __restrict__ sl_b, int* __restrict__ wfs_sym, int* __restrict__ sl_sym,
                                int* __restrict__ worst) {
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_tiles) return;
    wfs_sym[I] = wf_s[I] - sl_b[I];
    sl_sym[I] = sl_b[I] + sl_s[I];
    atomicMax(worst, sl_b[I] + sl_s[I]);
}

// 1 into *flag if the caller's events differ from the planned ones (bitwise)
__global__ void skip_same_events_kernel(int64_t m, const double* __restrict__ a, const double* __restrict__ b, int* flag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m && __double_as_longlong(a[i]) != __double_as_longlong(b[i])) *flag = 1;
}

// Cut a list (sorted by tile) into at most `workers` non-empty consecutive ranges of about equal cost.  The unit
// of the cut is a block of 32 streamed records, 4 per item (cost[k] is the cost of one block of item k): wstart
// (workers + 1 entries) is in blocks of the flattened (item, block) sequence; wfirst and slots are per tile.
// Returns the number of workers used.
int skip_cut(const std::vector<int2>& items, const std::vector<int>& cost, int n_tiles, int workers,
             std::vector<int>* wstart, std::vector<int>* wfirst, std::vector<int>* slots) {
    int64_t total = 0;
    for (int v : cost) total += 4 * (int64_t)v;
    const int64_t chunk = (total + workers - 1) / workers;
    wstart->assign(1, 0);
    wfirst->assign(n_tiles, 0);
    slots->assign(n_tiles, 0);
    std::vector<int> wlast(n_tiles, -1);
    int64_t acc = 0;
    int w = 0;
    const size_t nblocks = 4 * items.size();
    for (size_t q = 0; q < nblocks; ++q) {
        const int I = items[q / 4].x;
        if (wlast[I] < 0) (*wfirst)[I] = w;
        wlast[I] = w;
        acc += cost[q / 4];
        if (acc >= (int64_t)(w + 1) * chunk && q + 1 < nblocks) {
            ++w;
            wstart->push_back((int)q + 1);
        }
    }
    wstart->push_back((int)nblocks);
    for (int I = 0; I < n_tiles; ++I) (*slots)[I] = wlast[I] < 0 ? 0 : wlast[I] - (*wfirst)[I] + 1;
    return (int)wstart->size() - 1;
}

template <typename T>
int skip_upload(T** dst, const std::vector<T>& v) {
    *dst = nullptr;
    if (cudaMalloc((void**)dst, sizeof(T) * (v.size() ? v.size() : 1)) != cudaSuccess) return HAWKES_ERR_NOMEM;
    if (v.size() && cudaMemcpy(*dst, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice) != cudaSuccess)
        return HAWKES_ERR_CUDA;
    return HAWKES_OK;
}

int skip_build(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const hawkes_params* p, SkipPlan* old) {
    const int dim = ctx->dim, nd = dim + 1;   // axes: coordinates, then time
    SkipHost* hs = new (std::nothrow) SkipHost();
    if (!hs) return HAWKES_ERR_NOMEM;
    struct Guard { SkipHost*& h; ~Guard() { delete h; } } guard{hs};   // owned here until the plan takes it
    std::vector<double>&hx = hs->hx, &ht = hs->ht;
    // The caller's events (host or device pointers) are staged on the device: x, then t.  The new plan keeps this copy;
    // a later plan of the same events -- what an MCMC sweep asks for after every hyperparameter move -- recognises
    // them by a device-side comparison and never brings them to the host again.
    const size_t ev_doubles = (size_t)nd * (size_t)n;
    double* d_ev = nullptr;
    if (cudaMalloc((void**)&d_ev, ev_doubles * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return HAWKES_ERR_NOMEM; }
    struct EvGuard { double*& p; ~EvGuard() { if (p) cudaFree(p); } } ev_guard{d_ev};   // owned here until the plan takes it
    CK(cudaMemcpy(d_ev, x, sizeof(double) * dim * n, cudaMemcpyDefault));
    CK(cudaMemcpy(d_ev + (size_t)dim * n, t, sizeof(double) * n, cudaMemcpyDefault));
    auto val = [&](int a, int64_t i) { return a < dim ? hx[(size_t)a * n + i] : ht[i]; };

    // cut-off radii: a term is an exact zero beyond them whatever the other coordinates are
    const double inf = INFINITY;
    const double rs = p->h * std::sqrt(2.0 * SKIP_Z0), rb = p->tau_x * std::sqrt(2.0 * SKIP_Z0);
    const double ts_ = SKIP_Z0 / p->omega, tb = ctx->s_mode ? inf : p->tau_t * std::sqrt(2.0 * SKIP_Z0);
    // k-d order: split the events at a median of the axis along which they reach furthest in units of the cut-off
    // radius, the left part a whole number of tiles (of chunks, inside a tile), until every part is one chunk.
    // Tiles and chunks are then the leaves of the tree: compact boxes that end where the runs end.
    double cutoff[4] = {0, 0, 0, 0};
    for (int a = 0; a < nd; ++a) cutoff[a] = a < dim ? std::min(rs, rb) : std::min(ts_, tb);
    bool reuse = old && old->host && old->n == n && old->d_ev != nullptr && old->host->ht.size() == (size_t)n;
    for (int a = 0; a < nd && reuse; ++a) {
        const double r = cutoff[a] / old->host->cutoff[a];
        if (!(r >= 0.5 && r <= 2.0) && !(std::isinf(cutoff[a]) && std::isinf(old->host->cutoff[a]))) reuse = false;
    }
    if (reuse) {   // the same events, bit for bit?
        int* d_flag = reinterpret_cast<int*>(ctx->d_status + 1);   // status[1] is rewritten by the next evaluation's prep
        CK(cudaMemset(d_flag, 0, sizeof(int)));
        skip_same_events_kernel<<<(unsigned)((ev_doubles + 255) / 256), 256>>>((int64_t)ev_doubles, d_ev, old->d_ev, d_flag);
        int differ = 1;
        CK(cudaMemcpy(&differ, d_flag, sizeof(int), cudaMemcpyDeviceToHost));
        CK(cudaMemset(d_flag, 0, sizeof(int)));
        if (differ) reuse = false;
    }
    if (reuse) {
        hx.swap(old->host->hx);
        ht.swap(old->host->ht);
    } else {
        hx.resize((size_t)dim * n);
        ht.resize((size_t)n);
        CK(cudaMemcpy(hx.data(), d_ev, sizeof(double) * dim * n, cudaMemcpyDeviceToHost));
        CK(cudaMemcpy(ht.data(), d_ev + (size_t)dim * n, sizeof(double) * n, cudaMemcpyDeviceToHost));
        for (int64_t i = 0; i < n; ++i)
            if (!std::isfinite(ht[i])) return HAWKES_ERR_NONFINITE;
        for (size_t i = 0; i < hx.size(); ++i)
            if (!std::isfinite(hx[i])) return HAWKES_ERR_NONFINITE;
    }
    std::vector<int64_t>& perm = hs->perm;
    if (reuse) {
        perm.swap(old->host->perm);
        hs->chunk.swap(old->host->chunk);
        hs->tile.swap(old->host->tile);
        for (int a = 0; a < 4; ++a) hs->cutoff[a] = old->host->cutoff[a];
    } else {
        for (int a = 0; a < 4; ++a) hs->cutoff[a] = cutoff[a];
        perm.resize((size_t)n);
        for (int64_t i = 0; i < n; ++i) perm[i] = i;
        const int64_t tile = NT * P1_R;
        static_assert(NT * P1_R == NT * P2_R && (NT * P1_R) % TS == 0, "tiles of both passes are whole chunks");
        std::vector<std::pair<int64_t, int64_t>> stack(1, {0, n});
        while (!stack.empty()) {
            const int64_t b0 = stack.back().first, b1 = stack.back().second, len = b1 - b0;
            stack.pop_back();
            if (len <= TS) continue;
            int axis = 0;
            double best = -1.0;
            for (int a = 0; a < nd; ++a) {
                double lo = inf, hi = -inf;
                for (int64_t i = b0; i < b1; ++i) { lo = std::min(lo, val(a, perm[i])); hi = std::max(hi, val(a, perm[i])); }
                const double e = (hi - lo) / cutoff[a];
                if (e > best) { best = e; axis = a; }
            }
            const int64_t unit = len > tile ? tile : TS;
            int64_t nl = ((len + unit - 1) / unit / 2) * unit;
            if (nl <= 0) nl = unit;
            std::nth_element(perm.begin() + b0, perm.begin() + b0 + nl, perm.begin() + b1, [&](int64_t u, int64_t w) {
                const double vu = val(axis, u), vw = val(axis, w);
                return vu < vw || (vu == vw && u < w);
            });
            stack.push_back({b0, b0 + nl});
            stack.push_back({b0 + nl, b1});
        }
    }

    // boxes of the TS-record chunks and of the NT*R-record tiles
    auto boxes = [&](int run) {
        const int64_t nb = (n + run - 1) / run;
        std::vector<SkipBox> bx((size_t)nb);
        for (int64_t b = 0; b < nb; ++b) {
            for (int a = 0; a < 4; ++a) { bx[b].lo[a] = inf; bx[b].hi[a] = -inf; }
            for (int64_t i = b * run; i < std::min(n, (b + 1) * run); ++i)
                for (int a = 0; a < nd; ++a) {
                    const double v = val(a, perm[i]);
                    bx[b].lo[a] = std::min(bx[b].lo[a], v);
                    bx[b].hi[a] = std::max(bx[b].hi[a], v);
                }
        }
        return bx;
    };
    if (!reuse) {
        hs->chunk = boxes(TS);
        hs->tile = boxes(NT * P1_R);
    }
    const std::vector<SkipBox>&chunk = hs->chunk, &tile1 = hs->tile;

    SkipPlan* sp = new (std::nothrow) SkipPlan();
    if (!sp) return HAWKES_ERR_NOMEM;
    std::memset(sp, 0, sizeof(*sp));
    ctx->skip = sp;
    sp->host = hs;
    hs = nullptr;          // the plan owns it now (freed by skip_plan_free)
    sp->order_reused = reuse ? 1 : 0;
    sp->d_ev = d_ev;
    d_ev = nullptr;        // the plan owns the device copy of the events now
    sp->n = n;
    sp->p = *p;
    sp->s_mode = ctx->s_mode;
    const int nc = (int)chunk.size(), nt1 = (int)tile1.size(), nt2 = nt1;
    // ---- the four work lists and their cuts, all on the device (round 2; the host loops of round 1 took 39 ms per
    // re-plan at N = 250,000) ------------------------------------------------------------------------------------
    const int64_t ld = round_up(n, 256);
    const SkipGeom geom{dim, ctx->s_mode, p->tau_x, p->tau_t, p->h, p->omega};
    const int64_t np = (int64_t)nt1 * nt1;
    if (4 * np >= ((int64_t)1 << 31)) return HAWKES_ERR_UNSUPPORTED;
    struct DevTmp {
        void* p[8] = {};
        ~DevTmp() { for (void* q : p) if (q) cudaFree(q); }
    } tmp;
    auto dalloc = [&](int slot, void** dst, size_t bytes) {
        if (cudaMalloc(dst, bytes ? bytes : 8) != cudaSuccess) { cudaGetLastError(); *dst = nullptr; return false; }
        if (slot >= 0) tmp.p[slot] = *dst;
        return true;
    };
    SkipBox *d_tile = nullptr, *d_chunk = nullptr;
    int *d_cnt = nullptr, *d_off = nullptr;
    void* d_scan = nullptr;
    size_t scan_bytes = 0, scan_bytes64 = 0;
    cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, (const int*)nullptr, (int*)nullptr, (int)np);
    if (!dalloc(0, (void**)&d_tile, sizeof(SkipBox) * nt1) || !dalloc(1, (void**)&d_chunk, sizeof(SkipBox) * nc) ||
        !dalloc(2, (void**)&d_cnt, sizeof(int) * 4 * np) || !dalloc(3, (void**)&d_off, sizeof(int) * 4 * np) ||
        !dalloc(4, &d_scan, scan_bytes)) return HAWKES_ERR_NOMEM;
    CK(cudaMemcpy(d_tile, tile1.data(), sizeof(SkipBox) * nt1, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(d_chunk, chunk.data(), sizeof(SkipBox) * nc, cudaMemcpyHostToDevice));
    const unsigned gl = (unsigned)((np + 255) / 256);
    skip_lists_kernel<false><<<gl, 256>>>(nt1, nc, d_tile, d_chunk, geom, d_cnt, nullptr, nullptr, nullptr, nullptr, nullptr);
    for (int l = 0; l < 4; ++l)
        CK(cub::DeviceScan::ExclusiveSum(d_scan, scan_bytes, d_cnt + l * np, d_off + l * np, (int)np));
    int total[4];
    {
        int tails[8];   // last count and last offset of each list
        for (int l = 0; l < 4; ++l) {
            CK(cudaMemcpyAsync(&tails[2 * l], d_cnt + (l + 1) * np - 1, sizeof(int), cudaMemcpyDeviceToHost, 0));
            CK(cudaMemcpyAsync(&tails[2 * l + 1], d_off + (l + 1) * np - 1, sizeof(int), cudaMemcpyDeviceToHost, 0));
        }
        CK(cudaStreamSynchronize(0));
        for (int l = 0; l < 4; ++l) total[l] = tails[2 * l] + tails[2 * l + 1];
    }
    // the cut kernels index the quarter-blocks of a list as 4 * K in int (skip_cut_kernel, skip_compact_kernel, wstart)
    for (int l = 0; l < 4; ++l)
        if (total[l] < 0 || total[l] >= (1 << 29)) return HAWKES_ERR_UNSUPPORTED;
    // plan-owned pools: the items of the four lists; the cuts (ints)
    const int W1 = skip_sms(ctx) * P1_G[0], W2 = skip_sms(ctx) * P2_G[0], Wmax = std::max(W1, W2);
    int2* d_it[4];
    {
        size_t all = 0;
        for (int l = 0; l < 4; ++l) all += (size_t)total[l] + 1;
        if (!dalloc(-1, (void**)&sp->d_pool_items, sizeof(int2) * all)) return HAWKES_ERR_NOMEM;
        int2* base = sp->d_pool_items;
        for (int l = 0; l < 4; ++l) { d_it[l] = base; base += (size_t)total[l] + 1; }
    }
    const size_t per_list = (size_t)(Wmax + 1) + 3 * (size_t)nt1 + 1;     // wstart, tile_start, wfirst, slots
    const size_t pool_ints = 4 * per_list + 2 * (size_t)nt1 + 16;
    if (!dalloc(-1, (void**)&sp->d_pool_cut, sizeof(int) * pool_ints)) return HAWKES_ERR_NOMEM;
    int* cw[4]; int* ct[4]; int* cf[4]; int* cs[4];
    for (int l = 0; l < 4; ++l) {
        int* b0 = sp->d_pool_cut + l * per_list;
        cw[l] = b0; ct[l] = b0 + (Wmax + 1); cf[l] = ct[l] + nt1 + 1; cs[l] = cf[l] + nt1;
    }
    int* const d_wfs_sym = sp->d_pool_cut + 4 * per_list;
    int* const d_sl_sym = d_wfs_sym + nt1;
    int* const d_worst = d_sl_sym + nt1;                                  // + the count of B items (2 ints)
    skip_lists_kernel<true><<<gl, 256>>>(nt1, nc, d_tile, d_chunk, geom, nullptr, d_off, d_it[0], d_it[1], d_it[2], d_it[3]);
    CK(cudaGetLastError());
    // block costs of the pass-1 list (46 per background block, 37 per masked excitation block: DESIGN.md section 5's
    // issue model) and their prefix sums; the other lists have unit costs
    int* d_cost1 = nullptr;
    long long* d_C1 = nullptr;
    cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes64, (const int*)nullptr, (long long*)nullptr, total[0] + 1);
    void* d_scan64 = nullptr;
    if (!dalloc(5, (void**)&d_cost1, sizeof(int) * ((size_t)total[0] + 1)) ||
        !dalloc(6, (void**)&d_C1, sizeof(long long) * ((size_t)total[0] + 1)) || !dalloc(7, &d_scan64, scan_bytes64))
        return HAWKES_ERR_NOMEM;
    CK(cudaMemset(d_worst, 0, 4 * sizeof(int)));
    if (total[0] > 0) {
        skip_cost1_kernel<<<(unsigned)((total[0] + 255) / 256), 256>>>(total[0], d_it[0], W_ALL[1], W_HEAD[1] + 4, d_cost1,
                                                                      reinterpret_cast<unsigned long long*>(d_worst + 2));
        CK(cub::DeviceScan::ExclusiveSum(d_scan64, scan_bytes64, d_cost1, d_C1, total[0]));
    }
    // cut into workers; halve the worker count while the fullest tile's slots do not fit the partial buffers
    auto dcut = [&](int l, const int* cost, const long long* C, int workers, int n_mom, size_t cap, int* used) -> int {
        const int K = total[l], span = std::max(workers, nt1) + 1;
        for (;; workers = (workers + 1) / 2) {
            if (cudaMemset(d_worst, 0, sizeof(int)) != cudaSuccess) return HAWKES_ERR_CUDA;
            skip_cut_kernel<<<(unsigned)((span + 255) / 256), 256>>>(d_it[l], K, cost, C, workers, nt1, cw[l], ct[l]);
            skip_compact_kernel<<<1, 1>>>(workers, 4 * K, cw[l]);
            skip_slots_kernel<<<(unsigned)((nt1 + 255) / 256), 256>>>(nt1, workers, cw[l], ct[l], cf[l], cs[l], d_worst);
            int worst = 0;
            if (cudaMemcpy(&worst, d_worst, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return HAWKES_ERR_CUDA;
            if ((size_t)worst * n_mom * (size_t)ld <= cap) { *used = workers; return HAWKES_OK; }
            if (workers == 1) return HAWKES_ERR_UNSUPPORTED;
        }
    };
    int rc;
    if ((rc = dcut(0, d_cost1, d_C1, W1, 12, ctx->part1_doubles, &sp->workers1))) return rc;
    if ((rc = dcut(1, nullptr, nullptr, W1, 12, ctx->part1_doubles, &sp->workers1s))) return rc;
    if ((rc = dcut(3, nullptr, nullptr, W2, 2, ctx->part2_doubles, &sp->workers2))) return rc;
    sp->d_items1 = d_it[0]; sp->d_w1start = cw[0]; sp->d_w1first = cf[0]; sp->d_slots1 = cs[0];
    sp->d_items1s = d_it[1]; sp->d_w1sstart = cw[1]; sp->d_w1sfirst = cf[1]; sp->d_slots1s = cs[1];
    sp->d_items2 = d_it[3]; sp->d_w2start = cw[3]; sp->d_w2first = cf[3]; sp->d_slots2 = cs[3];
    sp->items_s = total[1];
    sp->items_p2 = total[3];
    sp->items_dense1 = (int64_t)nt1 * nc;
    sp->items_dense2 = (int64_t)nt2 * nc;
    {
        unsigned long long nb = 0;
        CK(cudaMemcpy(&nb, d_worst + 2, sizeof(nb), cudaMemcpyDeviceToHost));
        sp->items_b = (int64_t)nb;
    }
    {   // symmetric background: off unless it fits (hawkes_set_pass1_mode(DENSE) switches it off as in the dense path)
        sp->items_bsym = total[2];
        const int64_t Q = 4 * (int64_t)total[2];
        int Wb = 0, worst = 0;
        rc = Q > 0 ? dcut(2, nullptr, nullptr, W1, 0, (size_t)-1, &Wb) : HAWKES_OK;   // no capacity bound of its own ...
        if (rc) return rc;
        if (Q > 0) {                                                                  // ... the combined slots have
            CK(cudaMemset(d_worst, 0, sizeof(int)));
            skip_sym_kernel<<<(unsigned)((nt1 + 255) / 256), 256>>>(nt1, cf[1], cs[1], cs[2], d_wfs_sym, d_sl_sym, d_worst);
            CK(cudaMemcpy(&worst, d_worst, sizeof(int), cudaMemcpyDeviceToHost));
        }
        const size_t pcd = (size_t)colpart_doubles(nt1, NT * P1_R, 3);
        const size_t prd = (size_t)worst * 12 * (size_t)ld;
        // the two large buffers of the previous plan are taken over when they are large enough
        if (old && old->d_partc && old->partc_doubles >= pcd) {
            sp->d_partc = old->d_partc; sp->partc_doubles = old->partc_doubles;
            old->d_partc = nullptr;
        }
        if (old && old->d_part_sym && old->part_sym_doubles >= prd) {
            sp->d_part_sym = old->d_part_sym; sp->part_sym_doubles = old->part_sym_doubles;
            old->d_part_sym = nullptr;
        }
        if (!ctx->force_dense && Q > 0 && Q < ((int64_t)1 << 31) && prd * sizeof(double) <= ((size_t)8 << 30) &&
            pcd * sizeof(double) <= ((size_t)16 << 30) &&
            (sp->d_partc || cudaMalloc((void**)&sp->d_partc, pcd * sizeof(double)) == cudaSuccess) &&
            (sp->d_part_sym || cudaMalloc((void**)&sp->d_part_sym, prd * sizeof(double)) == cudaSuccess)) {
            if (!sp->partc_doubles) sp->partc_doubles = pcd;
            if (!sp->part_sym_doubles) sp->part_sym_doubles = prd;
            sp->partc_level = -1;
            sp->workersb = Wb;
            CK(cudaMemsetAsync(sp->d_partc, 0, sp->partc_doubles * sizeof(double), 0));
            sp->d_itemsb = d_it[2]; sp->d_wbstart = cw[2]; sp->d_wbfirst = cf[2];
            sp->d_w1sfirst_sym = d_wfs_sym; sp->d_slots_sym = d_sl_sym;
        } else {
            cudaGetLastError();
            if (sp->d_partc) cudaFree(sp->d_partc);
            sp->d_partc = nullptr;
        }
    }
    // the order on the device: taken over from the previous plan when it is the same
    if (reuse && old->d_perm) { sp->d_perm = old->d_perm; old->d_perm = nullptr; sp->d_tn = old->d_tn; old->d_tn = nullptr; }
    else {
        if ((rc = skip_upload(&sp->d_perm, perm))) return rc;
        double tn = -inf;
        for (int64_t i = 0; i < n; ++i) tn = std::max(tn, ht[i]);
        std::vector<double> tnv(1, tn);
        if ((rc = skip_upload(&sp->d_tn, tnv))) return rc;
    }
    CK(cudaDeviceSynchronize());
    return HAWKES_OK;
}

template <bool DIM3>
int enqueue_eval_skip(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                      const DevConsts& c, uint32_t want, double* ll, double* grad_theta, double* grad_hyper,
                      double* hess_theta_diag, double* hess_hyper, cudaStream_t st) {
    const SkipPlan& sp = *ctx->skip;
    const int level1 = (want & HAWKES_WANT_HESS_HYPER) ? 2 : ((want & HAWKES_WANT_GRAD_HYPER) ? 1 : 0);
    // background-sum cache of hawkes_hmc_run (LEVEL 0 only, record order of this plan): 1 = store, 2 = use; with the
    // cached sums pass 1 walks the list of the self-excitation items alone
    const int bg_mode = level1 == 0 ? ctx->bg_mode : 0;
    const bool s_only = bg_mode == 2;
    const bool sym = !s_only && level1 <= 1 && sp.d_partc != nullptr;   // background once per unordered pair
    const int64_t ld = round_up(n, 256);
    const int nblk = (int)((n + RED_T - 1) / RED_T);
    CK(cudaMemsetAsync(ctx->d_status, 0, 2 * sizeof(unsigned), st));
    skip_gather_kernel<<<nblk, RED_T, 0, st>>>(n, ctx->dim, sp.d_perm, x, t, theta, ctx->d_rec, ctx->d_status);
    Split s1{};
    s1.n = n;
    s1.tile = NT * P1_R;
    s1.n_tiles = (int)((n + s1.tile - 1) / s1.tile);
    s1.chunk = 1;
    s1.slot_tab = sym ? sp.d_slots_sym : (s_only ? sp.d_slots1s : sp.d_slots1);
    const int2* items1 = (s_only || sym) ? sp.d_items1s : sp.d_items1;
    const int* w1start = (s_only || sym) ? sp.d_w1sstart : sp.d_w1start;
    const int* w1first = sym ? sp.d_w1sfirst_sym : (s_only ? sp.d_w1sfirst : sp.d_w1first);
    const int workers1 = (s_only || sym) ? sp.workers1s : sp.workers1;
    const int nb1 = level1 == 0 ? 1 : 3;
    if (sym && ctx->skip->partc_level != nb1) {   // another moment layout: entries no item writes must read as zero
        if (ctx->skip->partc_level != -1) CK(cudaMemsetAsync(sp.d_partc, 0, sp.partc_doubles * sizeof(double), st));
        ctx->skip->partc_level = nb1;
    }
    const unsigned gb = (unsigned)((sp.workersb + P1_G[0] - 1) / P1_G[0]);
    double* const part1 = sym ? sp.d_part_sym : ctx->d_part1;
    constexpr int G1 = P1_G[0];
    constexpr unsigned SM1 = smem_request(G1 * group_buf_bytes<DIM3>());
    const unsigned g1 = (unsigned)((workers1 + G1 - 1) / G1);
#define SKIP_PASS1(L)                                                                                                     \
    if (sym) {                                                                                                            \
        pass1_symb_list_kernel<P1_R, (L) <= 1 ? (L) : 1, DIM3, G1>                                                        \
            <<<gb, NT * G1, smem_request(G1 * sym_group_bytes<DIM3>((L) == 0 ? 1 : 3)), st>>>(                            \
                ctx->d_rec, n, ld, c, ctx->d_tab, part1, sp.d_partc, s1.n_tiles, sp.d_itemsb, sp.d_wbstart,               \
                sp.d_wbfirst, sp.workersb);                                                                               \
        ctx->launches++;                                                                                                  \
    }                                                                                                                     \
    pass1_list_kernel<P1_R, L, DIM3, G1><<<g1, NT * G1, SM1, st>>>(ctx->d_rec, n, ld, c, ctx->d_tab, part1,              \
                                                                   items1, w1start, w1first, workers1);                   \
    reduce1_kernel<L, DIM3><<<nblk, RED_T, 0, st>>>(ctx->d_rec, n, ld, c, part1, s1, ctx->d_lam, ctx->d_trec,             \
                                                    ctx->d_trec2, (L) >= 1 ? ctx->d_rowd1 : nullptr, (L) >= 2 ? ctx->d_rowd2 : nullptr, nullptr, ctx->d_blockpart, ctx->d_status,               \
                                                    ctx->d_bgcache, bg_mode, sym ? sp.d_partc : nullptr, s1.n_tiles,      \
                                                    NT * P1_R, sp.d_tn)
    if (level1 == 0) { SKIP_PASS1(0); }
    else if (level1 == 1) { SKIP_PASS1(1); }
    else { SKIP_PASS1(2); }
#undef SKIP_PASS1
    ctx->launches += 3;
    // as in the dense path: the single-CTA scalar reduction runs on the side stream beside pass 2 when there is one
    const bool want_scal = (want & (HAWKES_WANT_LL | HAWKES_WANT_GRAD_HYPER | HAWKES_WANT_HESS_HYPER)) != 0;
    const bool scal_aside = want_scal && (want & (HAWKES_WANT_GRAD_THETA | HAWKES_WANT_HESS_THETA)) != 0;
    if (want_scal) {
        cudaStream_t ss = st;
        if (scal_aside) {
            CK(cudaEventRecord(ctx->ev_fork, st));
            CK(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
            ss = ctx->side;
        }
        scalars_kernel<<<1, SCAL_T, 0, ss>>>(ctx->d_blockpart, nblk, c, (want & HAWKES_WANT_LL) ? ll : nullptr,
                                             (want & HAWKES_WANT_GRAD_HYPER) ? grad_hyper : nullptr,
                                             (want & HAWKES_WANT_HESS_HYPER) ? hess_hyper : nullptr, ctx->d_scal);
        if (scal_aside) CK(cudaEventRecord(ctx->ev_join, ctx->side));
        ctx->launches++;
    }
    if (want & (HAWKES_WANT_GRAD_THETA | HAWKES_WANT_HESS_THETA)) {
        Split s2{};
        s2.n = n;
        s2.tile = NT * P2_R;
        s2.n_tiles = (int)((n + s2.tile - 1) / s2.tile);
        s2.chunk = 1;
        s2.slot_tab = sp.d_slots2;
        constexpr int G2 = P2_G[0];
        constexpr unsigned SM2 = smem_request(G2 * group_buf_bytes<DIM3>());
        const unsigned g2 = (unsigned)((sp.workers2 + G2 - 1) / G2);
        if (sp.items_p2 > 0) {
            if (want & HAWKES_WANT_HESS_THETA)
                pass2_list_kernel<P2_R, 1, DIM3, G2><<<g2, NT * G2, SM2, st>>>(ctx->d_rec, ctx->d_trec, n, ld, c, ctx->d_tab, ctx->d_part2, sp.d_items2, sp.d_w2start, sp.d_w2first, sp.workers2);
            else
                pass2_list_kernel<P2_R, 0, DIM3, G2><<<g2, NT * G2, SM2, st>>>(ctx->d_rec, ctx->d_trec, n, ld, c, ctx->d_tab, ctx->d_part2, sp.d_items2, sp.d_w2start, sp.d_w2first, sp.workers2);
            ctx->launches++;
        }
        theta_kernel<DIM3><<<nblk, RED_T, 0, st>>>(ctx->d_rec, n, ld, c, ctx->d_part2, s2,
                                                   (want & HAWKES_WANT_GRAD_THETA) ? grad_theta : nullptr,
                                                   (want & HAWKES_WANT_HESS_THETA) ? hess_theta_diag : nullptr, sp.d_tn,
                                                   sp.d_perm);
        ctx->launches++;
    }
    if (scal_aside) CK(cudaStreamWaitEvent(st, ctx->ev_join, 0));
    CK(cudaGetLastError());
    return HAWKES_OK;
}

template <bool DIM3>
int skip_setup_kernels() {
    int dummy;
    int rc;
    constexpr unsigned SM1 = smem_request(P1_G[0] * group_buf_bytes<DIM3>());
    constexpr unsigned SM2 = smem_request(P2_G[0] * group_buf_bytes<DIM3>());
    if ((rc = setup_kernel(pass1_list_kernel<P1_R, 0, DIM3, P1_G[0]>, P1_G[0], SM1, &dummy))) return rc;
    if ((rc = setup_kernel(pass1_list_kernel<P1_R, 1, DIM3, P1_G[0]>, P1_G[0], SM1, &dummy))) return rc;
    if ((rc = setup_kernel(pass1_list_kernel<P1_R, 2, DIM3, P1_G[0]>, P1_G[0], SM1, &dummy))) return rc;
    if ((rc = setup_kernel(pass1_symb_list_kernel<P1_R, 0, DIM3, P1_G[0]>, P1_G[0], smem_request(P1_G[0] * sym_group_bytes<DIM3>(1)), &dummy))) return rc;
    if ((rc = setup_kernel(pass1_symb_list_kernel<P1_R, 1, DIM3, P1_G[0]>, P1_G[0], smem_request(P1_G[0] * sym_group_bytes<DIM3>(3)), &dummy))) return rc;
    if ((rc = setup_kernel(pass2_list_kernel<P2_R, 0, DIM3, P2_G[0]>, P2_G[0], SM2, &dummy))) return rc;
    if ((rc = setup_kernel(pass2_list_kernel<P2_R, 1, DIM3, P2_G[0]>, P2_G[0], SM2, &dummy))) return rc;
    return HAWKES_OK;
}

}  // namespace

extern "C" {

int hawkes_skip_plan(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const hawkes_params* p) {
    if (!ctx || !x || !t || !p) return HAWKES_ERR_ARG;
    if (n < 1 || n > ctx->n_max) return HAWKES_ERR_ARG;
    DevConsts c;
    int rc = make_consts(p, ctx->dim, ctx->s_mode, &c);
    if (rc) return rc;
    CK(cudaSetDevice(ctx->device));
    CK(cudaDeviceSynchronize());   // evaluations in flight may still read the old plan
    SkipPlan* old = ctx->skip;     // detached: the new plan may take over its order, boxes and large buffers
    ctx->skip = nullptr;
    if (!old && (rc = (ctx->dim == 3 ? skip_setup_kernels<true>() : skip_setup_kernels<false>()))) return rc;
    rc = skip_build(ctx, n, x, t, p, old);
    if (rc) skip_plan_free(ctx);
    SkipPlan* fresh = ctx->skip;
    ctx->skip = old;
    skip_plan_free(ctx);           // what is left of the old plan
    ctx->skip = fresh;
    return rc;
}

int hawkes_eval_skip(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                     const hawkes_params* p, uint32_t want, double* ll, double* grad_theta, double* grad_hyper,
                     double* hess_theta_diag, double* hess_hyper, void* stream) {
    int rc = check_common(ctx, n, x, t, theta, p);
    if (rc) return rc;
    if (want == 0 || (want & ~31u)) return HAWKES_ERR_ARG;   // no cross block in this variant
    if (((want & HAWKES_WANT_LL) && !ll) || ((want & HAWKES_WANT_GRAD_THETA) && !grad_theta) ||
        ((want & HAWKES_WANT_GRAD_HYPER) && !grad_hyper) || ((want & HAWKES_WANT_HESS_THETA) && !hess_theta_diag) ||
        ((want & HAWKES_WANT_HESS_HYPER) && !hess_hyper))
        return HAWKES_ERR_ARG;
    const SkipPlan* sp = ctx->skip;
    if (!sp || sp->n != n || sp->s_mode != ctx->s_mode || sp->p.mu0 != p->mu0 || sp->p.tau_x != p->tau_x ||
        sp->p.tau_t != p->tau_t || sp->p.xi0 != p->xi0 || sp->p.h != p->h || sp->p.omega != p->omega)
        return HAWKES_ERR_ARG;     // no plan, or one built for other events / hyperparameters
    DevConsts c;
    rc = make_consts(p, ctx->dim, ctx->s_mode, &c);
    if (rc) return rc;
    CK(cudaSetDevice(ctx->device));
    if (ctx->dim == 3)
        return enqueue_eval_skip<true>(ctx, n, x, t, theta, c, want, ll, grad_theta, grad_hyper, hess_theta_diag, hess_hyper, (cudaStream_t)stream);
    return enqueue_eval_skip<false>(ctx, n, x, t, theta, c, want, ll, grad_theta, grad_hyper, hess_theta_diag, hess_hyper, (cudaStream_t)stream);
}

// out[0..4]: pass-1 items with a live background / with a live excitation / dense count; pass-2 items / dense count;
// out[5] = workers of pass 1, out[6] = workers of pass 2 (an item = NT*R records x TS records); out[7] = unordered
// background items of the symmetric form (0: not in use); out[8] = 1 if the order of the previous plan was kept
int hawkes_skip_stats(hawkes_ctx* ctx, int64_t* out) {
    if (!ctx || !out || !ctx->skip) return HAWKES_ERR_ARG;
    const SkipPlan* sp = ctx->skip;
    out[0] = sp->items_b; out[1] = sp->items_s; out[2] = sp->items_dense1;
    out[3] = sp->items_p2; out[4] = sp->items_dense2;
    out[5] = sp->workers1; out[6] = sp->workers2;
    out[7] = sp->d_partc ? sp->items_bsym : 0;
    out[8] = sp->order_reused;
    return HAWKES_OK;
}

int hawkes_skip_perm(hawkes_ctx* ctx, int64_t n, int64_t* perm_host) {
    if (!ctx || !perm_host || !ctx->skip || ctx->skip->n != n) return HAWKES_ERR_ARG;
    CK(cudaMemcpy(perm_host, ctx->skip->d_perm, sizeof(int64_t) * n, cudaMemcpyDeviceToHost));
    return HAWKES_OK;
}

}  // extern "C"
