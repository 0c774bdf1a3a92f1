// pass1_sym.cuh -- pass 1 with the background term evaluated once per UNORDERED pair (included by hawkes.cu inside
// its anonymous namespace; DESIGN.md section 5 "Symmetric background").
//
// B_{nn'} = B_{n'n}: the background exponential of the pair {n, n'} contributes the same three moments
// (e, e r^2, e dt^2) to the row sums of n and of n'.  The dense pass 1 evaluates it twice (N^2 exponentials); this
// kernel evaluates it once (N (N-1) / 2), together with the excitation term of the same pair (which only the later
// event receives), and accumulates
//   - the later event's six sums in registers (the thread owns R "target" events, as in the dense kernel), and
//   - the earlier event's three background sums in a COLUMN accumulator that travels with the streamed event:
//     a warp walks a block of 32 streamed events in 32 steps, lane l handling streamed event (l + s) & 31 at step s and
//     passing that event's column accumulator on to lane l - 1 by a shuffle, so that after 32 steps lane l holds the
//     column sums of event l over the warp's 32 R targets.  No cross-lane reduction tree, no atomics.
// The column sums of the four warps of a work group are combined in shared memory in warp order and written to the
// column partial of (target tile, streamed event): each element is written exactly once, and reduce1 adds an event's
// column partials in tile order => bit-identical results run to run.
//
// Streamed events sit in shared memory as SoA (x[TS], y[TS], [z[TS],] t[TS], w[TS]) so that the per-lane reads of 32
// consecutive (rotated) events are bank-conflict-free.

#ifndef HAWKES_SYM_UNROLL
#define HAWKES_SYM_UNROLL 2
#endif
constexpr int SYM_UNROLL = HAWKES_SYM_UNROLL;   // steps of the 32-step rotation unrolled together

// SoA tile: NA arrays of TS doubles
template <bool DIM3>
struct SoaIO {
    static constexpr int RS = DIM3 ? 6 : 4;
    static constexpr int NA = DIM3 ? 5 : 4;                 // arrays: x, y, (z,) t, w
    static constexpr int CH = RS / 2;
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
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int c = tid + q * NT, r = c / CH, part = c % CH;
            if (!DIM3) {                                    // (x, y) | (t, w)
                buf[(2 * part) * TS + r] = v[q].x;
                buf[(2 * part + 1) * TS + r] = v[q].y;
            } else {                                        // (x, y) | (z, t) | (w, 0)
                buf[(2 * part) * TS + r] = v[q].x;
                if (part < 2) buf[(2 * part + 1) * TS + r] = v[q].y;
            }
        }
    }
};

// one block of 32 streamed events (local indices j0 .. j0+31 of the tile in `sb`) against the warp's 32 R targets.
// MASKED: the pair (target gi[r], streamed event of global index jg0 + k) is evaluated iff k < nvalid and
// jg0 + k < gi[r] (index order: each unordered pair once, no self pair) -- plus, always, the paper's indicators
// (r2 != 0 for the background, dt > 0 for the excitation) and the underflow flush.
// S_ON = false: background only (the list-driven pass of skip.cuh, where the excitation term has its own items).
template <int R, int LEVEL, bool MASKED, bool DIM3, bool S_ON = true>
__device__ __forceinline__ void p1s_block(const double* __restrict__ sb, int j0, int nvalid, int64_t jg0,
                                          const Ev<DIM3> (&g)[R], const int64_t (&gi)[R], Mom<LEVEL> (&m)[R],
                                          double* __restrict__ colout /* this warp's [TS][NB] */, const P1C& c,
                                          unsigned lane_base, int lane) {
    constexpr int NB = Mom<LEVEL>::NB;
    constexpr int TO = DIM3 ? 3 : 2;        // array index of t
    constexpr int K = S_ON ? 2 * R : R;     // exponentials per step: background of the R pairs, then excitation
    double cc[NB];
#pragma unroll
    for (int k = 0; k < NB; ++k) cc[k] = 0.0;
    int idx = lane;
    const int src = (lane + 1) & 31;
#pragma unroll ((LEVEL == 0 || !S_ON) ? 4 : SYM_UNROLL)   // level 0: 0.686 -> 0.656 ms at N=23,422 with 4; level 1: 2 (4: 0.757 against 0.733)
    for (int s = 0; s < 32; ++s) {
        const double* p = sb + j0 + idx;
        Ev<DIM3> e;
        e.x = p[0]; e.y = p[TS]; e.z = DIM3 ? p[2 * TS] : 0.0; e.t = p[TO * TS]; e.w = p[(TO + 1) * TS];
        // The shuffles below make ptxas treat this loop as possibly divergent, and it then keeps the loop constants
        // in vector registers: a Horner step would read three of them.  The K exponentials of a step are therefore
        // evaluated in lockstep, stage by stage, so that consecutive FP64 instructions share the constant (and negc)
        // in the same operand slot and hit the operand-reuse cache (2 fresh registers each: DESIGN.md section 5).
        double u[R], w[R], dt[R], a[2 * R], t[2 * R], f[2 * R], q[2 * R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double dx = g[r].x - e.x, dy = g[r].y - e.y;
            dt[r] = g[r].t - e.t;
            u[r] = fma(dy, dy, dx * dx);
            if (DIM3) { const double dz = g[r].z - e.z; u[r] = fma(dz, dz, u[r]); }
            w[r] = dt[r] * dt[r];
        }
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = fma(c.rho_b, w[r], u[r]);
        if (S_ON) {
#pragma unroll
            for (int r = 0; r < R; ++r) a[R + r] = fma(c.rho_s, dt[r], u[r]);
        }
#pragma unroll
        for (int i = 0; i < K; ++i) t[i] = fma(a[i], i < R ? c.negcb : c.negcs, c.e.magic);
#pragma unroll
        for (int i = 0; i < K; ++i) f[i] = t[i] - c.e.magic;
#pragma unroll
        for (int i = 0; i < K; ++i) f[i] = fma(a[i], i < R ? c.negcb : c.negcs, -f[i]);
#pragma unroll
        for (int i = 0; i < K; ++i) q[i] = f[i] + c.e.d3;
#pragma unroll
        for (int i = 0; i < K; ++i) q[i] = fma(q[i], f[i], c.e.d2);
#pragma unroll
        for (int i = 0; i < K; ++i) q[i] = fma(q[i], f[i], c.e.d1);
#pragma unroll
        for (int i = 0; i < K; ++i) q[i] = fma(q[i], f[i], c.e.d0);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double eB, eS = 0.0;
            if (MASKED) {
                const int live = (idx < nvalid && jg0 + idx < gi[r]) ? 1 : 0;
                eB = exp2_table<4>(a[r], t[r], c.lim_b_hi, u[r], lane_base, live) * q[r];
                if (S_ON) eS = exp2_table<5>(a[R + r], t[R + r], c.lim_s_hi, dt[r], lane_base, live) * q[R + r];
            } else {
                eB = exp2_table<1>(a[r], t[r], c.lim_b_hi, u[r], lane_base) * q[r];
                if (S_ON) eS = exp2_table<0>(a[R + r], t[R + r], c.lim_s_hi, dt[r], lane_base) * q[R + r];
            }
            if (S_ON) eS *= e.w;
            m[r].b[0] += eB;
            cc[0] += eB;
            if (S_ON) m[r].s[0] += eS;
            if (LEVEL == 1) {
                m[r].b[1] = fma(eB, u[r], m[r].b[1]);
                cc[1 % NB] = fma(eB, u[r], cc[1 % NB]);
                m[r].b[2] = fma(eB, w[r], m[r].b[2]);
                cc[2 % NB] = fma(eB, w[r], cc[2 % NB]);
                if (S_ON) {
                    m[r].s[1] = fma(eS, u[r], m[r].s[1]);
                    m[r].s[2] = fma(eS, dt[r], m[r].s[2]);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NB; ++k)   // in place: the accumulator keeps its register pair across the rotation
            asm volatile("{\n\t.reg .b32 lo, hi;\n\tmov.b64 {lo, hi}, %0;\n\t"
                         "shfl.sync.idx.b32 lo, lo, %1, 0x1f, 0xffffffff;\n\t"
                         "shfl.sync.idx.b32 hi, hi, %1, 0x1f, 0xffffffff;\n\tmov.b64 %0, {lo, hi};\n\t}"
                         : "+d"(cc[k]) : "r"(src));
        idx = (idx + 1) & 31;
    }
    // lane l now holds the column sums of streamed event j0 + l
#pragma unroll
    for (int k = 0; k < NB; ++k) colout[(j0 + lane) * NB + k] = cc[k];
}

// column partial of (target tile I, streamed event j): slot s = I - j / tile; slot s holds NB rows of
// len(s) = (n_tiles - s) * tile doubles, slots stored back to back (a triangle, N^2 NB / (2 tile) doubles in all)
__host__ __device__ inline int64_t colpart_index(int n_tiles, int tile, int nb, int s, int k, int64_t j) {
    const int64_t off = (int64_t)nb * tile * ((int64_t)s * n_tiles - (int64_t)s * (s - 1) / 2);
    const int64_t len = (int64_t)(n_tiles - s) * tile;
    return off + (int64_t)k * len + j;
}
__host__ __device__ inline int64_t colpart_doubles(int n_tiles, int tile, int nb) {
    return (int64_t)nb * tile * ((int64_t)n_tiles * (n_tiles + 1) / 2);
}

template <bool DIM3> constexpr unsigned sym_group_bytes(int nb) {
    return (unsigned)((2 * SoaIO<DIM3>::NA * TS + (NT / 32) * TS * nb) * sizeof(double));
}

// Work decomposition: Split with w_all = 0 (tile I streams the events [0, end of tile I)), one segment per worker
// as in the dense kernel.  part: row partials [(slot*2NB + k)*ld + i]; partc: column partials (colpart_index).
#ifdef HAWKES_SYM_MAXREG
#define HAWKES_SYM_BOUNDS __maxnreg__(HAWKES_SYM_MAXREG)
#else
#define HAWKES_SYM_BOUNDS __launch_bounds__(NT * G, 1)
#endif
template <int R, int LEVEL, bool DIM3, int G>
__global__ void HAWKES_SYM_BOUNDS pass1s_kernel(const double* __restrict__ rec, int64_t n, int64_t ld,
                                                           DevConsts c, const double* __restrict__ tab_g,
                                                           double* __restrict__ part, double* __restrict__ partc, Split sp) {
    constexpr int RS = DIM3 ? 6 : 4;
    constexpr int TOFF = DIM3 ? 3 : 2;
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
    const int64_t vcta = (int64_t)blockIdx.x * G + grp + sp.w_begin;
    double* const gbuf = reinterpret_cast<double*>(smem + plan.buf_off + grp * GB);
    double* const sbuf0 = gbuf;
    double* const sbuf1 = gbuf + NA * TS;
    double* const colacc = gbuf + 2 * NA * TS;            // [NT/32][TS][NB]
    double* const mycol = colacc + wrp * TS * NB;
    const unsigned lane_base = (smem_base + plan.tab_off) | (8u * lane);

    const int64_t total = split_prefix(sp, sp.n_tiles);
    const int64_t lo = vcta * sp.chunk;
    if (lo >= total || vcta >= sp.w_end) return;
    const int64_t hi = min(lo + sp.chunk, total);
    // every loop constant through shared memory: held in vector registers, never re-loaded inside the loops
    P1C pc;
    {
        const volatile P1C& v = spc;
        pc.negcb = v.negcb; pc.negcs = v.negcs; pc.rho_b = v.rho_b; pc.rho_s = v.rho_s;
        pc.lim_b_hi = v.lim_b_hi; pc.lim_s_hi = v.lim_s_hi;
        pc.e.d0 = v.e.d0; pc.e.d1 = v.e.d1; pc.e.d2 = v.e.d2; pc.e.d3 = v.e.d3; pc.e.magic = v.e.magic;
    }

    for (int I = split_tile_of(sp, lo); I < sp.n_tiles; ++I) {
        const int64_t base = split_prefix(sp, I);
        if (base >= hi) break;
        const int64_t cost_I = split_prefix(sp, I + 1) - base;
        const int64_t jb = split_pos(sp, I, max(lo - base, (int64_t)0));
        const int64_t je = split_pos(sp, I, min(hi - base, cost_I));
        const int64_t i0 = (int64_t)I * (NT * R);
        const int64_t i1 = min(i0 + (int64_t)NT * R, n);
        const bool ragged_tile = i1 - i0 < NT * R;

        Ev<DIM3> g[R];
        int64_t gi[R];
        Mom<LEVEL> m[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = i0 + r * NT + tid;
            gi[r] = i < n ? i : -1;                      // a target past the end owns no pair
            g[r] = read_rec<DIM3>(rec + min(i, n - 1) * RS);
#pragma unroll
            for (int k = 0; k < NB; ++k) { m[r].b[k] = 0.0; m[r].s[k] = 0.0; }
        }
        const double t_first = rec[i0 * RS + TOFF];   // earliest target time of this tile

        SoaIO<DIM3> io;
        int64_t a = jb;
        int64_t b = min(je, (a / TS + 1) * TS);
        group_sync(grp);
        if (a < je) {
            io.load(rec, a, (int)(b - a), tid);
            io.store(sbuf0, tid);
        }
        group_sync(grp);
        int cur = 0;
        while (a < je) {
            const int cnt = (int)(b - a);
            const int64_t a2 = b, b2 = min(je, b + TS);
            if (a2 < je) io.load(rec, a2, (int)(b2 - a2), tid);
            const double* sb = cur ? sbuf1 : sbuf0;
            // every pair of an off-diagonal piece is causal in index; it is causal in time too unless a tie
            // straddles the tile boundary
            const bool plain = !ragged_tile && b <= i0 && rec[(b - 1) * RS + TOFF] < t_first;
            for (int j0 = 0; j0 < cnt; j0 += 32) {
                const int nvalid = min(32, cnt - j0);
                if (plain && nvalid == 32)
                    p1s_block<R, LEVEL, false, DIM3>(sb, j0, nvalid, a + j0, g, gi, m, mycol, pc, lane_base, lane);
                else
                    p1s_block<R, LEVEL, true, DIM3>(sb, j0, nvalid, a + j0, g, gi, m, mycol, pc, lane_base, lane);
            }
            if (a2 < je) io.store(cur ? sbuf0 : sbuf1, tid);
            group_sync(grp);
            // column sums of this piece: the four warps' shares in warp order, one streamed event per thread
            if (tid < cnt) {
                const int64_t j = a + tid;
                const int s = I - (int)(j / (NT * R));
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    double v = 0.0;
#pragma unroll
                    for (int w = 0; w < NT / 32; ++w) v += colacc[(w * TS + tid) * NB + k];
                    partc[colpart_index(sp.n_tiles, NT * R, NB, s, k, j)] = v;
                }
            }
            group_sync(grp);
            cur ^= 1;
            a = a2;
            b = b2;
        }
        const int slot = split_slot_of(sp, vcta, base);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = i0 + r * NT + tid;
            if (i < n) {
                double* o = part + (int64_t)slot * (2 * NB) * ld + i;
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    o[(int64_t)k * ld] = m[r].b[k];
                    o[(int64_t)(NB + k) * ld] = m[r].s[k];
                }
            }
        }
    }
}
