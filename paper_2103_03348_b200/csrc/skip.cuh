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

void skip_plan_free(hawkes_ctx* c) {
    SkipPlan* s = c->skip;
    if (!s) return;
    void* ptrs[] = {s->d_perm, s->d_tn, s->d_items1, s->d_w1start, s->d_w1first, s->d_slots1,
                    s->d_items1s, s->d_w1sstart, s->d_w1sfirst, s->d_slots1s, s->d_itemsb, s->d_wbstart, s->d_wbfirst,
                    s->d_w1sfirst_sym, s->d_slots_sym, s->d_partc, s->d_part_sym, s->d_items2, s->d_w2start, s->d_w2first, s->d_slots2};
    for (void* q : ptrs)
        if (q) cudaFree(q);
    delete s->host;
    delete s;
    c->skip = nullptr;
}

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
    hx.resize((size_t)dim * n);
    ht.resize((size_t)n);
    CK(cudaMemcpy(hx.data(), x, sizeof(double) * dim * n, cudaMemcpyDefault));
    CK(cudaMemcpy(ht.data(), t, sizeof(double) * n, cudaMemcpyDefault));
    for (int64_t i = 0; i < n; ++i)
        if (!std::isfinite(ht[i])) return HAWKES_ERR_NONFINITE;
    for (size_t i = 0; i < hx.size(); ++i)
        if (!std::isfinite(hx[i])) return HAWKES_ERR_NONFINITE;
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
    bool reuse = old && old->host && old->n == n && old->host->hx.size() == hx.size() &&
                 std::memcmp(old->host->hx.data(), hx.data(), hx.size() * sizeof(double)) == 0 &&
                 std::memcmp(old->host->ht.data(), ht.data(), ht.size() * sizeof(double)) == 0;
    for (int a = 0; a < nd && reuse; ++a) {
        const double r = cutoff[a] / old->host->cutoff[a];
        if (!(r >= 0.5 && r <= 2.0) && !(std::isinf(cutoff[a]) && std::isinf(old->host->cutoff[a]))) reuse = false;
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
    const std::vector<SkipBox>&chunk = hs->chunk, &tile1 = hs->tile, &tile2 = hs->tile;
    auto gap2 = [&](const SkipBox& A, const SkipBox& B) {   // squared distance between the spatial boxes
        double s = 0.0;
        for (int a = 0; a < dim; ++a) {
            const double g = std::max(0.0, std::max(A.lo[a] - B.hi[a], B.lo[a] - A.hi[a]));
            s += g * g;
        }
        return s;
    };
    // background of (targets T, sources S): min exponent r^2/2tau_x^2 + dt^2/2tau_t^2
    auto live_b = [&](const SkipBox& T, const SkipBox& S) {
        double z = gap2(T, S) / (2.0 * p->tau_x * p->tau_x);
        if (!ctx->s_mode) {
            const double g = std::max(0.0, std::max(T.lo[dim] - S.hi[dim], S.lo[dim] - T.hi[dim]));
            z += g * g / (2.0 * p->tau_t * p->tau_t);
        }
        return !(z >= SKIP_Z0);
    };
    // excitation of targets T by sources S: some pair must be causal (t_n > t_m), min exponent r^2/2h^2 + omega dt
    auto live_s = [&](const SkipBox& T, const SkipBox& S) {
        if (!(T.hi[dim] > S.lo[dim])) return false;
        const double z = gap2(T, S) / (2.0 * p->h * p->h) + p->omega * std::max(0.0, T.lo[dim] - S.hi[dim]);
        return !(z >= SKIP_Z0);
    };

    SkipPlan* sp = new (std::nothrow) SkipPlan();
    if (!sp) return HAWKES_ERR_NOMEM;
    std::memset(sp, 0, sizeof(*sp));
    ctx->skip = sp;
    sp->host = hs;
    hs = nullptr;          // the plan owns it now (freed by skip_plan_free)
    sp->order_reused = reuse ? 1 : 0;
    sp->n = n;
    sp->p = *p;
    sp->s_mode = ctx->s_mode;
    const int nc = (int)chunk.size(), nt1 = (int)tile1.size(), nt2 = (int)tile2.size();
    std::vector<int2> items1, items1s, items2;
    std::vector<int> cost1, cost1s, cost2;
    // a chunk's box lies inside its tile's: a pair of tiles that is dead leaves nothing to test below it
    constexpr int CPT = (NT * P1_R) / TS;   // chunks per tile
    for (int I = 0; I < nt1; ++I)
        for (int Jt = 0; Jt < nt1; ++Jt) {
            const bool tb_live = live_b(tile1[I], tile1[Jt]), ts_live = live_s(tile1[I], tile1[Jt]);
            if (!tb_live && !ts_live) continue;
            for (int J = Jt * CPT; J < std::min(nc, (Jt + 1) * CPT); ++J) {
            const int kind = ((tb_live && live_b(tile1[I], chunk[J])) ? SK_B : 0) |
                             ((ts_live && live_s(tile1[I], chunk[J])) ? SK_S : 0);
            if (!kind) continue;
            items1.push_back(make_int2(I, J * 4 + kind));
            cost1.push_back(((kind & SK_B) ? W_ALL[1] : 0) + ((kind & SK_S) ? W_HEAD[1] + 4 : 0));
            sp->items_b += (kind & SK_B) ? 1 : 0;
            sp->items_s += (kind & SK_S) ? 1 : 0;
            if (kind & SK_S) {
                items1s.push_back(make_int2(I, J * 4 + SK_S));
                cost1s.push_back(1);
            }
            }
        }
    for (int M = 0; M < nt2; ++M)
        for (int Jt = 0; Jt < nt2; ++Jt) {
            if (!live_s(tile2[Jt], tile2[M])) continue;
            for (int J = Jt * CPT; J < std::min(nc, (Jt + 1) * CPT); ++J)
                if (live_s(chunk[J], tile2[M])) {
                    items2.push_back(make_int2(M, J * 4 + SK_S));
                    cost2.push_back(1);
                }
        }
    sp->items_p2 = (int64_t)items2.size();
    sp->items_dense1 = (int64_t)nt1 * nc;
    sp->items_dense2 = (int64_t)nt2 * nc;

    // cut into workers; halve the worker count while the fullest tile's slots do not fit the partial buffers
    const int64_t ld = round_up(n, 256);
    std::vector<int> ws, wf, sl;
    auto cut = [&](const std::vector<int2>& items, const std::vector<int>& cost, int n_tiles, int workers, int n_mom,
                   size_t cap, int* used) {
        for (;; workers = (workers + 1) / 2) {
            *used = skip_cut(items, cost, n_tiles, workers, &ws, &wf, &sl);
            int worst = 0;
            for (int v : sl) worst = std::max(worst, v);
            if ((size_t)worst * n_mom * (size_t)ld <= cap) return HAWKES_OK;
            if (workers == 1) return HAWKES_ERR_UNSUPPORTED;
        }
    };
    int rc;
    if ((rc = cut(items1, cost1, nt1, skip_sms(ctx) * P1_G[0], 12, ctx->part1_doubles, &sp->workers1))) return rc;
    if ((rc = skip_upload(&sp->d_items1, items1)) || (rc = skip_upload(&sp->d_w1start, ws)) ||
        (rc = skip_upload(&sp->d_w1first, wf)) || (rc = skip_upload(&sp->d_slots1, sl))) return rc;
    if ((rc = cut(items1s, cost1s, nt1, skip_sms(ctx) * P1_G[0], 12, ctx->part1_doubles, &sp->workers1s))) return rc;
    if ((rc = skip_upload(&sp->d_items1s, items1s)) || (rc = skip_upload(&sp->d_w1sstart, ws)) ||
        (rc = skip_upload(&sp->d_w1sfirst, wf)) || (rc = skip_upload(&sp->d_slots1s, sl))) return rc;
    {   // symmetric background: off unless it fits (hawkes_set_pass1_mode(DENSE) switches it off as in the dense path)
        const std::vector<int> wf_s = wf, sl_s = sl;          // cut of the S items, just made
        std::vector<int2> itemsb;
        for (int I = 0; I < nt1; ++I)
            for (int Jt = 0; Jt <= I; ++Jt) {
                if (!live_b(tile1[I], tile1[Jt])) continue;
                for (int J = Jt * CPT; J < std::min(nc, (Jt + 1) * CPT); ++J)
                    if (live_b(tile1[I], chunk[J])) itemsb.push_back(make_int2(I, J));
            }
        sp->items_bsym = (int64_t)itemsb.size();
        const int64_t Q = 4 * (int64_t)itemsb.size();
        const int W = (int)std::min<int64_t>(skip_sms(ctx) * P1_G[0], Q);
        std::vector<int> wb(W + 1), wbf(nt1, 0), slb(nt1, 0), wbl(nt1, -1);
        for (int w = 0; w <= W; ++w) wb[w] = (int)(Q * w / W);
        for (int w = 0; w < W; ++w)
            for (int k = wb[w] / 4; k <= (wb[w + 1] - 1) / 4 && wb[w] < wb[w + 1]; ++k) {
                const int I = itemsb[k].x;
                if (wbl[I] < 0) wbf[I] = w;
                wbl[I] = w;
            }
        int worst = 0;
        std::vector<int> wfs_sym(nt1), sl_sym(nt1);
        for (int I = 0; I < nt1; ++I) {
            slb[I] = wbl[I] < 0 ? 0 : wbl[I] - wbf[I] + 1;
            wfs_sym[I] = wf_s[I] - slb[I];
            sl_sym[I] = slb[I] + sl_s[I];
            worst = std::max(worst, sl_sym[I]);
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
            sp->workersb = W;
            CK(cudaMemset(sp->d_partc, 0, sp->partc_doubles * sizeof(double)));
            if ((rc = skip_upload(&sp->d_itemsb, itemsb)) || (rc = skip_upload(&sp->d_wbstart, wb)) ||
                (rc = skip_upload(&sp->d_wbfirst, wbf)) || (rc = skip_upload(&sp->d_w1sfirst_sym, wfs_sym)) ||
                (rc = skip_upload(&sp->d_slots_sym, sl_sym))) return rc;
        } else {
            cudaGetLastError();
            if (sp->d_partc) cudaFree(sp->d_partc);
            sp->d_partc = nullptr;
        }
    }
    if ((rc = cut(items2, cost2, nt2, skip_sms(ctx) * P2_G[0], 2, ctx->part2_doubles, &sp->workers2))) return rc;
    if ((rc = skip_upload(&sp->d_items2, items2)) || (rc = skip_upload(&sp->d_w2start, ws)) ||
        (rc = skip_upload(&sp->d_w2first, wf)) || (rc = skip_upload(&sp->d_slots2, sl))) return rc;
    if ((rc = skip_upload(&sp->d_perm, perm))) return rc;
    double tn = -inf;
    for (int64_t i = 0; i < n; ++i) tn = std::max(tn, ht[i]);
    std::vector<double> tnv(1, tn);
    if ((rc = skip_upload(&sp->d_tn, tnv))) return rc;
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
