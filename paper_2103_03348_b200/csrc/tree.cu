// tree.cu -- O(M) evaluation of the phylogenetic Brownian-diffusion prior on the log-rates z (section 2.2,
// Eq. 2) and of its z-gradient, for sm_100a.  Contract: include/hawkes.h (hawkes_tree_*); design: DESIGN.md section 11.
//
// PAPER.md:121 cites the linear-time dynamic programme (post-order message passing on the tree) without printing
// it; what is implemented is the independent-contrasts recursion, which factorises Eq. 2 exactly:
//   every node carries the message (m, v): the value of the process at that node is, given the tips below it,
//   normal with mean m and variance sigma^2 v.   Tips: (z_i, 0).   Internal node u with children a, b:
//     v_a' = v_a + w_a,  v_b' = v_b + w_b,  c = m_a - m_b,  s = v_a' + v_b'
//     log p += -1/2 [ log(2 pi sigma^2 s) + c^2 / (sigma^2 s) ]          (the contrast c ~ N(0, sigma^2 s))
//     alpha = v_b' / s,  m_u = alpha m_a + (1 - alpha) m_b,  v_u = v_a' v_b' / s
//   root:  s = v_root + tau0,  c = m_root,  same term                     (root value ~ N(0, tau0 sigma^2))
//   M terms in all (M - 1 internal nodes + the root), matching (2 pi sigma^2)^(-M/2) |V_G|^(-1/2) of Eq. 2.
// Gradient by one reverse sweep (adjoint of m):  mbar_root = -m_root / (sigma^2 s_root);
//   mbar_a = alpha mbar_u - c / (sigma^2 s),  mbar_b = (1 - alpha) mbar_u + c / (sigma^2 s);  d log p / d z_i = mbar_tip_i.
//
// One CTA walks the tree level by level (level = height above the deepest tip below; all nodes of a level are
// independent), the node messages living in shared memory (two doubles per node) when the tree fits, else in a
// global scratch.  Sums are accumulated per thread over a fixed node assignment and reduced in a fixed order, so
// results are bit-identical run to run.
#include "../../include/hawkes.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <new>
#include <vector>

namespace {

constexpr int TREE_T = 1024;
constexpr size_t TREE_SMEM_MAX = 200 * 1024;

#define CKT(call)                                          \
    do {                                                   \
        if ((call) != cudaSuccess) return HAWKES_ERR_CUDA; \
    } while (0)

// an internal node in level order: its id, its children, alpha_u and 1 / s_u of the up sweep
struct __align__(16) TreeQ {
    int u, a, b, pad;
    double alpha, inv;
};

// fixed-order block sum of two values; result in thread 0
__device__ __forceinline__ void block_sum2(double& a, double& b, double* red /*[2 * TREE_T / 32]*/) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, off);
        b += __shfl_down_sync(0xffffffffu, b, off);
    }
    if (lane == 0) { red[2 * wid] = a; red[2 * wid + 1] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0.0, sb = 0.0;
        for (int w = 0; w < TREE_T / 32; ++w) { sa += red[2 * w]; sb += red[2 * w + 1]; }
        a = sa; b = sb;
    }
}

// The message variances, hence s_u, alpha_u and sum log s_u, depend on the branch lengths alone: hawkes_tree_create
// computes them once on the host (alpha[q], inv[q] = 1 / s_u by level-order position q, the sum of log s_u and the
// root's message variance), and a call walks the means only -- no division and no logarithm on the per-level
// critical path.
// node storage: nm[v], nv[v] (v = node id).  Life of the slots of the children a, b of an internal node u:
//   up sweep, before u:   nm = message mean
//   up sweep, after u:    nm[b] = c_u / (sigma^2 s_u)   (the messages of a, b are dead)
//   down sweep:           nv[a], nv[b] = adjoints mbar_a, mbar_b
template <bool SMEM>
__global__ void __launch_bounds__(TREE_T) tree_prior_kernel(int n_tips, int n_levels, int narrow_from,
                                                            const int* __restrict__ g_level_start,
                                                            const TreeQ* __restrict__ g_tq, double logs_tree, double v_root,
                                                            int root, const double* __restrict__ z, double sigma2,
                                                            double tau0, double* __restrict__ scratch,
                                                            double* __restrict__ logp, double* __restrict__ grad_z) {
    extern __shared__ __align__(16) double sm[];
    __shared__ double red[2 * TREE_T / 32];
    const int n_nodes = 2 * n_tips - 1, n_int = n_tips - 1;
    double* nm = SMEM ? sm : scratch;
    double* nv = nm + n_nodes;
    // topology in level order (position q = 0 .. M-2): node id, children, the children's branch lengths.  With SMEM
    // it is copied next to the messages so that a level costs shared-memory latency only.
    const TreeQ* tq = g_tq;
    const int* level_start = g_level_start;
    if (SMEM) {
        TreeQ* s_tq = reinterpret_cast<TreeQ*>(nv + n_nodes);   // 32-byte records: two 16-byte loads per node
        int* s_ls = reinterpret_cast<int*>(s_tq + n_int);
        for (int q = threadIdx.x; q < n_int; q += TREE_T) s_tq[q] = g_tq[q];
        for (int l = threadIdx.x; l <= n_levels; l += TREE_T) s_ls[l] = g_level_start[l];
        tq = s_tq; level_start = s_ls;
    }
    // z == NULL (SMEM only, one CTA per tip): z = the unit vector of tip blockIdx.x; the gradient goes to row blockIdx.x
    // of grad_z -- the rows of -V_G^-1 / sigma^2, the Hessian of the quadratic log prior (tree_dense_* below)
    for (int i = threadIdx.x; i < n_tips; i += TREE_T) nm[i] = z ? z[i] : (i == (int)blockIdx.x ? 1.0 : 0.0);
    if (!z) grad_z += (size_t)blockIdx.x * n_tips;
    __syncthreads();
    const double inv_s2 = 1.0 / sigma2;
    double quad = 0.0;
    // up sweep: levels 1 .. n_levels (level_start has n_levels + 1 entries; entry l-1 .. l bound level l).
    // Levels below `narrow_from` are walked by the whole CTA with a block barrier each; from `narrow_from` on every
    // level has at most 32 nodes and warp 0 walks them alone, one warp barrier per level.
    auto up_node = [&](int q) {
        const TreeQ r = tq[q];
        const double ma = nm[r.a], mb = nm[r.b];
        const double c = ma - mb;
        nm[r.u] = fma(r.alpha, c, mb);      // alpha ma + (1 - alpha) mb
        quad = fma(c * c, r.inv, quad);
        nm[r.b] = c * r.inv * inv_s2;
    };
    for (int l = 0; l < narrow_from; ++l) {
        for (int q = level_start[l] + threadIdx.x; q < level_start[l + 1]; q += TREE_T) up_node(q);
        __syncthreads();
    }
    if (threadIdx.x < 32) {
        for (int l = narrow_from; l < n_levels; ++l) {
            const int q = level_start[l] + threadIdx.x;
            if (q < level_start[l + 1]) up_node(q);
            __syncwarp();
        }
    }
    __syncthreads();
    // sum of log s over the internal nodes: a constant of the tree; the root term holds tau0
    double logs = 0.0;
    double mbar_root = 0.0;
    if (threadIdx.x == 0) {
        const double s = v_root + tau0, c = nm[root];
        quad = fma(c * c, 1.0 / s, quad);
        logs = logs_tree + log(s);
        mbar_root = -c / (sigma2 * s);
    }
    __syncthreads();
    if (threadIdx.x == 0) nv[root] = mbar_root;
    block_sum2(quad, logs, red);   // contains a barrier: nv[root] is visible after it
    if (threadIdx.x == 0 && logp)
        *logp = -0.5 * ((double)n_tips * log(6.283185307179586476925286766559 * sigma2) + logs + quad * inv_s2);
    if (grad_z == nullptr) return;
    // down sweep (narrow levels first, by warp 0)
    auto down_node = [&](int q) {
        const TreeQ r = tq[q];
        const double mbar = nv[r.u], k = nm[r.b];
        nv[r.a] = fma(r.alpha, mbar, -k);
        nv[r.b] = fma(1.0 - r.alpha, mbar, k);
    };
    if (threadIdx.x < 32) {
        for (int l = n_levels - 1; l >= narrow_from; --l) {
            const int q = level_start[l] + threadIdx.x;
            if (q < level_start[l + 1]) down_node(q);
            __syncwarp();
        }
    }
    __syncthreads();
    for (int l = narrow_from - 1; l >= 0; --l) {
        for (int q = level_start[l] + threadIdx.x; q < level_start[l + 1]; q += TREE_T) down_node(q);
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n_tips; i += TREE_T) grad_z[i] = nv[i];
}

// diag(V_G^-1) / sigma^2 by two sweeps over variances only: v_up[u] = variance of the message of u's subtree,
// v_out[u] = variance of u's value given every tip OUTSIDE its subtree (root: tau0, the root prior); for a tip,
// v_out is its conditional variance given all other tips (in units of sigma^2), whose reciprocal is the
// diagonal entry of the precision matrix.  Run once per tree / (sigma^2, tau0): node store in global scratch.
__global__ void __launch_bounds__(TREE_T) tree_precision_kernel(int n_tips, int n_levels, const int* __restrict__ level_start,
                                                                const int* __restrict__ order, const int* __restrict__ child_a,
                                                                const int* __restrict__ child_b, const double* __restrict__ branch,
                                                                int root, double sigma2, double tau0, double* __restrict__ scratch,
                                                                double* __restrict__ prec_diag) {
    const int n_nodes = 2 * n_tips - 1;
    double* vup = scratch;
    double* vout = scratch + n_nodes;
    for (int i = threadIdx.x; i < n_tips; i += TREE_T) vup[i] = 0.0;
    __syncthreads();
    for (int l = 0; l < n_levels; ++l) {
        for (int q = level_start[l] + threadIdx.x; q < level_start[l + 1]; q += TREE_T) {
            const int u = order[q], a = child_a[u], b = child_b[u];
            const double va = vup[a] + branch[a], vb = vup[b] + branch[b];
            vup[u] = va * vb / (va + vb);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) vout[root] = tau0;
    __syncthreads();
    for (int l = n_levels - 1; l >= 0; --l) {
        for (int q = level_start[l] + threadIdx.x; q < level_start[l + 1]; q += TREE_T) {
            const int u = order[q], a = child_a[u], b = child_b[u];
            const double va = vup[a] + branch[a], vb = vup[b] + branch[b], o = vout[u];
            vout[a] = ((o + vb > 0.0) ? o * vb / (o + vb) : 0.0) + branch[a];
            vout[b] = ((o + va > 0.0) ? o * va / (o + va) : 0.0) + branch[b];
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n_tips; i += TREE_T) prec_diag[i] = 1.0 / (sigma2 * vout[i]);
}

// The log prior is quadratic: log p(z) = log p(0) + 1/2 z^T G z with G = -V_G^-1 / sigma^2, grad = G z.  For the variants of
// hawkes_hmc_run that cache every constant of a call (the kernel matrix), G is formed once (its rows are the gradients
// at the unit vectors: M CTAs of tree_prior_kernel) and a prior evaluation becomes one dense symmetric matrix-vector
// product out of L2 (20 MB at M = 1,610) instead of a latency-bound walk of the tree's ~150 levels.
// One warp per row, lane-strided, fixed shuffle tree: bit-identical run to run.
constexpr int DENSE_ROWS = 8;   // rows (warps) per CTA
__global__ void __launch_bounds__(32 * DENSE_ROWS) tree_dense_gemv_kernel(int m, const double* __restrict__ G,
                                                                          const double* __restrict__ z,
                                                                          double* __restrict__ grad, double* __restrict__ zy) {
    const int row = blockIdx.x * DENSE_ROWS + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= m) return;
    const double* g = G + (size_t)row * m;
    double a = 0.0;
    for (int k = lane; k < m; k += 32) a = fma(g[k], z[k], a);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) a += __shfl_down_sync(0xffffffffu, a, off);
    if (lane == 0) {
        if (grad) grad[row] = a;
        zy[row] = z[row] * a;
    }
}
// log p = log p(0) + 1/2 sum_i z_i (G z)_i: one CTA, thread j takes i = j, j + 1024, ..., then a fixed tree
__global__ void __launch_bounds__(1024) tree_dense_logp_kernel(int m, const double* __restrict__ zy, double logp0,
                                                               double* __restrict__ logp) {
    __shared__ double red[32];
    double a = 0.0;
    for (int i = threadIdx.x; i < m; i += 1024) a += zy[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) a += __shfl_down_sync(0xffffffffu, a, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double r = 0.0;
        for (int w = 0; w < 32; ++w) r += red[w];
        *logp = logp0 + 0.5 * r;
    }
}

}  // namespace

struct hawkes_tree {
    int device;
    int n_tips, n_levels, narrow_from, root;
    int *d_level_start, *d_order, *d_child_a, *d_child_b;   // child_a/b: by node id (precision kernel)
    TreeQ* d_tq;                                            // prior kernel: one record per internal node, level order
    double logs_tree, v_root;                               // sum log s_u over the internal nodes; the root's message variance
    double *d_branch, *d_scratch;
    bool smem;
    size_t smem_bytes;
    int64_t launches;
    double* d_G;          // dense -V_G^-1 / sigma^2 (tree_dense_*), built on first use for (G_sigma2, G_tau0), or NULL
    double* d_zy;         // M products z_i (G z)_i + 1
    double G_sigma2, G_tau0, G_logp0;
};

extern "C" {

int hawkes_tree_create(hawkes_tree** out, int32_t n_tips, const int32_t* parent, const double* branch, int device) {
    if (!out || !parent || !branch || n_tips < 1) return HAWKES_ERR_ARG;
    const int M = n_tips, nn = 2 * M - 1;
    std::vector<int> ca(nn, -1), cb(nn, -1), level(nn, 0), pending(nn, 0);
    int root = -1;
    for (int v = 0; v < nn; ++v) {
        const int p = parent[v];
        if (p < 0) {
            if (root >= 0) return HAWKES_ERR_ARG;   // two roots
            root = v;
            continue;
        }
        if (p >= nn || p < M || p == v) return HAWKES_ERR_ARG;          // parents are internal nodes
        if (!(branch[v] >= 0.0) || !std::isfinite(branch[v])) return HAWKES_ERR_ARG;
        if (ca[p] < 0) ca[p] = v;
        else if (cb[p] < 0) cb[p] = v;
        else return HAWKES_ERR_ARG;                                      // more than two children
    }
    if (root < 0) return HAWKES_ERR_ARG;
    for (int v = M; v < nn; ++v)
        if (ca[v] < 0 || cb[v] < 0) return HAWKES_ERR_ARG;               // internal node without two children
    // levels by peeling: a node is ready when both children are done (detects cycles / disconnected parts)
    std::vector<int> ready;
    for (int v = 0; v < M; ++v) ready.push_back(v);
    size_t head = 0;
    int done = 0, n_levels = 0;
    while (head < ready.size()) {
        const int v = ready[head++];
        ++done;
        const int p = parent[v];
        if (p < 0) continue;
        level[p] = level[p] > level[v] + 1 ? level[p] : level[v] + 1;
        if (++pending[p] == 2) ready.push_back(p);
    }
    if (done != nn) return HAWKES_ERR_ARG;
    for (int v = M; v < nn; ++v) n_levels = level[v] > n_levels ? level[v] : n_levels;
    std::vector<int> level_start(n_levels + 1, 0), order(M > 1 ? M - 1 : 1, 0);
    for (int v = M; v < nn; ++v) level_start[level[v]]++;       // count per level l at index l (levels 1..n_levels)
    // prefix: level l occupies [start[l-1], start[l])
    {
        std::vector<int> cnt(level_start);
        int acc = 0;
        level_start[0] = 0;
        for (int l = 1; l <= n_levels; ++l) { acc += cnt[l]; level_start[l] = acc; }
        std::vector<int> fill(n_levels + 1, 0);
        for (int v = M; v < nn; ++v) {
            const int l = level[v];
            order[level_start[l - 1] + fill[l]++] = v;
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return HAWKES_ERR_CUDA;
    CKT(cudaSetDevice(device));
    hawkes_tree* t = new (std::nothrow) hawkes_tree();
    if (!t) return HAWKES_ERR_NOMEM;
    t->device = device; t->n_tips = M; t->n_levels = n_levels; t->root = root; t->launches = 0;
    t->d_G = nullptr; t->d_zy = nullptr; t->G_sigma2 = t->G_tau0 = t->G_logp0 = 0.0;
    // first level from which every level holds at most 32 nodes (walked by a single warp)
    t->narrow_from = n_levels;
    while (t->narrow_from > 0 && level_start[t->narrow_from] - level_start[t->narrow_from - 1] <= 32) t->narrow_from--;
    // shared memory of the prior kernel: 2 message doubles per node + per internal node 2 doubles and 3 ints + the level offsets
    t->smem_bytes = sizeof(double) * 2 * (size_t)nn + (size_t)(M - 1) * sizeof(TreeQ) +
                    (size_t)(n_levels + 1) * sizeof(int) + 16;
    std::vector<int> qa(M > 1 ? M - 1 : 1, 0), qb(M > 1 ? M - 1 : 1, 0);
    std::vector<double> qwa(M > 1 ? M - 1 : 1, 0.0), qwb(M > 1 ? M - 1 : 1, 0.0);
    // variance half of the independent-contrasts recursion: it involves the branch lengths only
    std::vector<double> hv(nn, 0.0);
    double logs_tree = 0.0;
    for (int q = 0; q < M - 1; ++q) {
        const int u = order[q];
        qa[q] = ca[u]; qb[q] = cb[u];
        const double va = hv[ca[u]] + branch[ca[u]], vb = hv[cb[u]] + branch[cb[u]];
        const double sm_ = va + vb, inv = 1.0 / sm_;
        qwa[q] = vb * inv;       // alpha_u
        qwb[q] = inv;            // 1 / s_u
        hv[u] = va * vb * inv;
        logs_tree += std::log(sm_);
    }
    t->logs_tree = logs_tree;
    t->v_root = hv[root];
    std::vector<TreeQ> tqv(M > 1 ? M - 1 : 1);
    for (int q = 0; q < M - 1; ++q) tqv[q] = TreeQ{order[q], qa[q], qb[q], 0, qwa[q], qwb[q]};
    t->smem = t->smem_bytes <= TREE_SMEM_MAX;
    t->d_level_start = t->d_order = t->d_child_a = t->d_child_b = nullptr;
    t->d_tq = nullptr;
    t->d_branch = t->d_scratch = nullptr;
    bool ok = true;
    auto up = [&](void** d, const void* h, size_t bytes) {
        if (!ok) return;
        if (cudaMalloc(d, bytes ? bytes : 8) != cudaSuccess) { ok = false; *d = nullptr; return; }
        if (h && bytes && cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) != cudaSuccess) ok = false;
    };
    up((void**)&t->d_level_start, level_start.data(), sizeof(int) * level_start.size());
    up((void**)&t->d_order, order.data(), sizeof(int) * order.size());
    up((void**)&t->d_child_a, ca.data(), sizeof(int) * nn);
    up((void**)&t->d_child_b, cb.data(), sizeof(int) * nn);
    up((void**)&t->d_branch, branch, sizeof(double) * nn);
    up((void**)&t->d_tq, tqv.data(), sizeof(TreeQ) * tqv.size());
    up((void**)&t->d_scratch, nullptr, sizeof(double) * 2 * (size_t)nn);
    if (ok && t->smem &&
        cudaFuncSetAttribute(tree_prior_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->smem_bytes) != cudaSuccess)
        ok = false;
    if (!ok) {
        hawkes_tree_destroy(t);
        cudaGetLastError();
        return HAWKES_ERR_NOMEM;
    }
    *out = t;
    return HAWKES_OK;
}

void hawkes_tree_destroy(hawkes_tree* t) {
    if (!t) return;
    cudaSetDevice(t->device);
    void* ptrs[] = {t->d_level_start, t->d_order, t->d_child_a, t->d_child_b, t->d_branch, t->d_scratch,
                    t->d_tq, t->d_G, t->d_zy};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    delete t;
}

int hawkes_tree_prior(hawkes_tree* t, const double* z, double sigma2, double tau0, double* logp, double* grad_z,
                      void* stream) {
    if (!t || !z || (!logp && !grad_z)) return HAWKES_ERR_ARG;
    if (!(sigma2 > 0.0) || !std::isfinite(sigma2) || !(tau0 >= 0.0) || !std::isfinite(tau0)) return HAWKES_ERR_PARAM;
    CKT(cudaSetDevice(t->device));
    cudaStream_t st = (cudaStream_t)stream;
    if (t->smem)
        tree_prior_kernel<true><<<1, TREE_T, t->smem_bytes, st>>>(t->n_tips, t->n_levels, t->narrow_from, t->d_level_start,
                                                                 t->d_tq, t->logs_tree, t->v_root,
                                                                 t->root, z, sigma2, tau0, t->d_scratch, logp, grad_z);
    else
        tree_prior_kernel<false><<<1, TREE_T, 0, st>>>(t->n_tips, t->n_levels, t->narrow_from, t->d_level_start,
                                                       t->d_tq, t->logs_tree, t->v_root, t->root, z, sigma2,
                                                       tau0, t->d_scratch, logp, grad_z);
    t->launches++;
    CKT(cudaGetLastError());
    return HAWKES_OK;
}

int hawkes_tree_precision_diag(hawkes_tree* t, double sigma2, double tau0, double* prec_diag, void* stream) {
    if (!t || !prec_diag) return HAWKES_ERR_ARG;
    if (!(sigma2 > 0.0) || !std::isfinite(sigma2) || !(tau0 >= 0.0) || !std::isfinite(tau0)) return HAWKES_ERR_PARAM;
    CKT(cudaSetDevice(t->device));
    tree_precision_kernel<<<1, TREE_T, 0, (cudaStream_t)stream>>>(t->n_tips, t->n_levels, t->d_level_start, t->d_order,
                                                                 t->d_child_a, t->d_child_b, t->d_branch, t->root, sigma2,
                                                                 tau0, t->d_scratch, prec_diag);
    t->launches++;
    CKT(cudaGetLastError());
    return HAWKES_OK;
}

int32_t hawkes_tree_levels(const hawkes_tree* t) { return t ? t->n_levels : 0; }
int64_t hawkes_tree_launch_count(const hawkes_tree* t) { return t ? t->launches : 0; }

/* Internal (hawkes_hmc_run, cached-matrix variants; not part of the C ABI).  hk_tree_dense_prepare: forms G for
 * (sigma2, tau0) unless the tree holds it already; may allocate M x M doubles and synchronises `stream` once (log p(0)).
 * HAWKES_ERR_UNSUPPORTED if the tree does not fit shared memory (M > ~3,100): the caller then walks the tree.
 * hk_tree_dense_prior: log p(z) into *logp (may be NULL) and G z into grad_z (may be NULL), enqueued on `stream`. */
int hk_tree_dense_prepare(hawkes_tree* t, double sigma2, double tau0, void* stream) {
    if (!t || !(sigma2 > 0.0) || !std::isfinite(sigma2) || !(tau0 >= 0.0) || !std::isfinite(tau0)) return HAWKES_ERR_PARAM;
    if (!t->smem) return HAWKES_ERR_UNSUPPORTED;
    if (t->d_G && t->G_sigma2 == sigma2 && t->G_tau0 == tau0) return HAWKES_OK;
    CKT(cudaSetDevice(t->device));
    cudaStream_t st = (cudaStream_t)stream;
    const int M = t->n_tips;
    if (!t->d_G) {
        if (cudaMalloc((void**)&t->d_G, sizeof(double) * (size_t)M * M) != cudaSuccess ||
            cudaMalloc((void**)&t->d_zy, sizeof(double) * ((size_t)M + 1)) != cudaSuccess) {
            cudaGetLastError();
            if (t->d_G) cudaFree(t->d_G);
            t->d_G = nullptr;
            return HAWKES_ERR_NOMEM;
        }
    }
    tree_prior_kernel<true><<<M, TREE_T, t->smem_bytes, st>>>(t->n_tips, t->n_levels, t->narrow_from, t->d_level_start, t->d_tq,
                                                             t->logs_tree, t->v_root, t->root, nullptr, sigma2, tau0,
                                                             t->d_scratch, nullptr, t->d_G);
    // log p(0): the kernel at z = 0 (d_zy serves as the zero vector, then receives the scalar)
    CKT(cudaMemsetAsync(t->d_zy, 0, sizeof(double) * ((size_t)M + 1), st));
    tree_prior_kernel<true><<<1, TREE_T, t->smem_bytes, st>>>(t->n_tips, t->n_levels, t->narrow_from, t->d_level_start, t->d_tq,
                                                             t->logs_tree, t->v_root, t->root, t->d_zy, sigma2, tau0,
                                                             t->d_scratch, t->d_zy + M, nullptr);
    t->launches += 2;
    CKT(cudaMemcpyAsync(&t->G_logp0, t->d_zy + M, sizeof(double), cudaMemcpyDeviceToHost, st));
    CKT(cudaStreamSynchronize(st));
    CKT(cudaGetLastError());
    t->G_sigma2 = sigma2;
    t->G_tau0 = tau0;
    return HAWKES_OK;
}

int hk_tree_dense_prior(hawkes_tree* t, const double* z, double* logp, double* grad_z, void* stream) {
    if (!t || !t->d_G || !z) return HAWKES_ERR_ARG;
    CKT(cudaSetDevice(t->device));
    cudaStream_t st = (cudaStream_t)stream;
    const int M = t->n_tips;
    tree_dense_gemv_kernel<<<(unsigned)((M + DENSE_ROWS - 1) / DENSE_ROWS), 32 * DENSE_ROWS, 0, st>>>(M, t->d_G, z, grad_z, t->d_zy);
    t->launches++;
    if (logp) {
        tree_dense_logp_kernel<<<1, 1024, 0, st>>>(M, t->d_zy, t->G_logp0, logp);
        t->launches++;
    }
    CKT(cudaGetLastError());
    return HAWKES_OK;
}

/* Counts kernels of this tree that ran inside a replayed CUDA graph (hawkes_hmc_run launches them k at a time). */
void hk_tree_count_launches(hawkes_tree* t, int64_t k) { if (t) t->launches += k; }

}  // extern "C"
