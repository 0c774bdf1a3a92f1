// ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain definition of the phylogenetic Brownian-diffusion prior on the log-rates z (section 2.2):
//
//   V_G = {v_nm}:  v_mm = tau0 + d_F(root, tip m)
//                  v_nm = tau0 + [ d_F(root, tip n) + d_F(root, tip m) - d_F(tip n, tip m) ] / 2
//                  d_F(u, v) = sum of edge weights along the path between u and v in the tree
//   log p(z | V_G, sigma^2, tau0) = -M/2 log(2 pi sigma^2) - 1/2 log|V_G| - z^T V_G^-1 z / (2 sigma^2)   (Eq. 2, l.101)
//   d log p / d z = - V_G^-1 z / sigma^2
//
// written out densely: path sums for every pair of tips, then a Cholesky factorisation V_G = L L^T in long
// double.  O(M^2 depth) + O(M^3); it is the thing the O(M) message-passing kernel of the CUDA path
// (PAPER.md:121 cites it, does not print it) must reproduce.  Shares nothing with paper_2103_03348_b200/csrc/.
//
// Tree encoding (same as include/hawkes.h): 2M-1 nodes; nodes 0..M-1 are the tips (tip i carries z[i]);
// parent[v] is the parent node of v, parent[root] = -1; branch[v] = edge weight w_v between v and parent[v]
// (branch[root] is ignored).
//
// Pins: tests/test_tree_pins.py (M = 1 and M = 2 closed forms; a hand-written 4-tip V_G; the joint Gaussian of
// all 2M-1 node values built from the generative description at PAPER.md:99 and marginalised to the tips;
// star-tree Sherman-Morrison closed form; central finite differences of the gradient).
#include <cmath>
#include <cstdint>
#include <vector>

namespace {

typedef long double ld;

// depth-first distance of every node from the root; returns the root (or -1 if the encoding is broken)
int64_t root_distances(int64_t n_nodes, const int32_t* parent, const double* branch, std::vector<ld>& dist,
                       std::vector<int32_t>& depth) {
    dist.assign(n_nodes, 0.0L);
    depth.assign(n_nodes, 0);
    int64_t root = -1;
    for (int64_t v = 0; v < n_nodes; ++v) {
        if (parent[v] < 0) {
            if (root >= 0) return -1;
            root = v;
        }
    }
    if (root < 0) return -1;
    for (int64_t v = 0; v < n_nodes; ++v) {
        ld d = 0.0L;
        int32_t k = 0;
        int64_t u = v;
        while (parent[u] >= 0) {
            d += (ld)branch[u];
            u = parent[u];
            if (++k > n_nodes) return -1;   // cycle
        }
        dist[v] = d;
        depth[v] = k;
    }
    return root;
}

}  // namespace

extern "C" {

// V_out[M*M] row-major (double).  Returns 0, or -1 on a malformed tree.
int tree_ref_vg(int32_t n_tips, const int32_t* parent, const double* branch, double tau0, double* V_out) {
    const int64_t M = n_tips, n_nodes = 2 * M - 1;
    if (M < 1) return -1;
    std::vector<ld> dist;
    std::vector<int32_t> depth;
    if (root_distances(n_nodes, parent, branch, dist, depth) < 0) return -1;
    for (int64_t i = 0; i < M; ++i) {
        for (int64_t j = i; j < M; ++j) {
            // d_F(tip i, tip j): walk both tips up to their meeting point, adding the edges passed
            int64_t a = i, b = j;
            ld dij = 0.0L;
            while (a != b) {
                if (depth[a] >= depth[b]) { dij += (ld)branch[a]; a = parent[a]; }
                else { dij += (ld)branch[b]; b = parent[b]; }
            }
            const ld v = (ld)tau0 + (dist[i] + dist[j] - dij) / 2.0L;
            V_out[i * M + j] = (double)v;
            V_out[j * M + i] = (double)v;
        }
    }
    return 0;
}

// Eq. 2 and its z-gradient from a dense V (row-major M*M doubles).  Returns 0; 1 if V is not positive definite
// (logp = NaN).  grad may be NULL.
int tree_ref_logp(int32_t n_tips, const double* V, const double* z, double sigma2, double* logp, double* grad) {
    const int64_t M = n_tips;
    std::vector<ld> L((size_t)M * M, 0.0L);
    ld logdet = 0.0L;
    for (int64_t j = 0; j < M; ++j) {
        ld s = (ld)V[j * M + j];
        for (int64_t k = 0; k < j; ++k) s -= L[j * M + k] * L[j * M + k];
        if (!(s > 0.0L)) { *logp = NAN; return 1; }
        const ld d = sqrtl(s);
        L[j * M + j] = d;
        logdet += 2.0L * logl(d);
        for (int64_t i = j + 1; i < M; ++i) {
            ld r = (ld)V[i * M + j];
            for (int64_t k = 0; k < j; ++k) r -= L[i * M + k] * L[j * M + k];
            L[i * M + j] = r / d;
        }
    }
    // y = L^-1 z ;  z^T V^-1 z = |y|^2 ;  V^-1 z = L^-T y
    std::vector<ld> y(M);
    ld quad = 0.0L;
    for (int64_t i = 0; i < M; ++i) {
        ld r = (ld)z[i];
        for (int64_t k = 0; k < i; ++k) r -= L[i * M + k] * y[k];
        y[i] = r / L[i * M + i];
        quad += y[i] * y[i];
    }
    const ld two_pi = 6.283185307179586476925286766559005768L;
    *logp = (double)(-0.5L * (ld)M * logl(two_pi * (ld)sigma2) - 0.5L * logdet - quad / (2.0L * (ld)sigma2));
    if (grad) {
        std::vector<ld> x(M);
        for (int64_t i = M - 1; i >= 0; --i) {
            ld r = y[i];
            for (int64_t k = i + 1; k < M; ++k) r -= L[k * M + i] * x[k];
            x[i] = r / L[i * M + i];
        }
        for (int64_t i = 0; i < M; ++i) grad[i] = (double)(-x[i] / (ld)sigma2);
    }
    return 0;
}

// diag(V^-1) / sigma2 = - d2 log p / d z_m^2 (the prior's own curvature; used as the constant part of the HMC
// preconditioner, reading R6): dense, from the Cholesky factor: (V^-1)_ii = sum_k (L^-1)_ki^2.
int tree_ref_precision_diag(int32_t n_tips, const double* V, double sigma2, double* out) {
    const int64_t M = n_tips;
    std::vector<ld> L((size_t)M * M, 0.0L);
    for (int64_t j = 0; j < M; ++j) {
        ld s = (ld)V[j * M + j];
        for (int64_t k = 0; k < j; ++k) s -= L[j * M + k] * L[j * M + k];
        if (!(s > 0.0L)) return 1;
        const ld d = sqrtl(s);
        L[j * M + j] = d;
        for (int64_t i = j + 1; i < M; ++i) {
            ld r = (ld)V[i * M + j];
            for (int64_t k = 0; k < j; ++k) r -= L[i * M + k] * L[j * M + k];
            L[i * M + j] = r / d;
        }
    }
    std::vector<ld> col(M);
    for (int64_t i = 0; i < M; ++i) {
        // column i of L^-1: solve L y = e_i
        ld acc = 0.0L;
        for (int64_t r = i; r < M; ++r) {
            ld v = (r == i) ? 1.0L : 0.0L;
            for (int64_t k = i; k < r; ++k) v -= L[r * M + k] * col[k];
            col[r] = v / L[r * M + r];
            acc += col[r] * col[r];
        }
        out[i] = (double)(acc / (ld)sigma2);
    }
    return 0;
}

}  // extern "C"
