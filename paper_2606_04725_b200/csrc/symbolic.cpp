// symbolic.cpp -- host-once symbolic analysis (step a0).  See symbolic.h.  Integer work only; no CUDA.
#include "symbolic.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <functional>
#include <numeric>
#include <queue>

namespace nmpc {

void default_options(nmpc_options* o) {
    std::memset(o, 0, sizeof(*o));
    o->ordering = NMPC_ORDER_AUTO;
    o->nd_leaf = 0;                // 0 = choose from the structure
    o->relax_small = -1;           // auto: nmpc_analyze uses 64, or 32 for small (latency-mode) problems; the host-only nmpc_symbolic_analyze 8
    o->relax_zeros = 0.05;         // fraction-based merging lengthens the fronts at the top of the tree (the critical path): keep it small
    o->smem_front_max = 0;         // 0 = device default
    o->use_graph = 1;
    // IPM constants: readings S0 of DESIGN.md section 3 (the paper prints none)
    o->gamma = 1e-4; o->eps_outer = 1e-5; o->mu0 = 0.1; o->mu_warm = 0.0 /* -> eps_outer/10 */;
    o->kappa_eps = 10.0; o->kappa_mu = 0.2; o->theta_mu = 1.5; o->tau_min = 0.99;
    o->kappa_push = 1e-2; o->s_floor = 1e-2; o->s_max = 100.0; o->max_iter = 200;
    o->eta_first = 1e-4; o->eta_grow_first = 100.0; o->eta_grow = 8.0; o->eta_shrink = 1.0 / 3.0;
    o->eta_min = 1e-20; o->eta_max = 1e40; o->warm_push = 1e-10;
    // globalisation / refinement (off): constants of ref. [17] as recalled, proposals like the S0 constants
    o->refine_steps = 0; o->globalization = 0;
    o->gamma_theta = 1e-5; o->gamma_phi = 1e-8; o->delta_sw = 1.0; o->s_theta = 1.1; o->s_phi = 2.3; o->eta_phi = 1e-8;
    o->theta_max_fact = 1e4; o->theta_min_fact = 1e-4; o->ls_max_backtracks = 30;
    o->gamma_h = 1e6; o->cg_tol = 1e-10; o->cg_max_iter = 50;     // HyKKT (reading G21)
    o->fuse_rhs = -1;              // auto: the right-hand-side row is carried through the factorization when the handle has a model
}

// =============================================================================================================
// Model patterns and gather maps
// =============================================================================================================
bool build_model_maps(const nmpc_ocp* ocp, ModelMaps& mm, std::string& err) {
    if (!ocp || ocp->model == NMPC_MODEL_NONE) { mm.present = false; return true; }
    ModelDesc& D = mm.desc;
    D.model = ocp->model; D.N = ocp->N; D.nx = ocp->nx; D.nu = ocp->nu; D.nr = ocp->nr; D.nv = ocp->nx + ocp->nu;
    D.dt = ocp->dt;
    if (D.N < 1 || D.nx < 1 || D.nu < 0) { err = "bad OCP sizes"; return false; }
    if (ocp->n_model_params > 12 || ocp->n_model_params < 0 || (ocp->n_model_params && !ocp->model_params)) {
        err = "bad model_params"; return false;
    }
    for (int i = 0; i < 12; ++i) D.p[i] = i < ocp->n_model_params ? ocp->model_params[i] : 0.0;
    switch (D.model) {
        case MODEL_VDP:
            if (D.nx != 2 || D.nu != 1 || D.nr != 2 || ocp->n_model_params < 2) { err = "VDP: nx=2,nu=1,nr=2, 2 params"; return false; }
            break;
        case MODEL_DISTILL:
            if (D.nx < 3 || D.nu != 1 || D.nr != 1 || ocp->n_model_params < 10) { err = "DISTILL: nx>=3,nu=1,nr=1, 10 params"; return false; }
            if ((int)D.p[7] < 1 || (int)D.p[7] > D.nx - 2) { err = "DISTILL: feed index out of range"; return false; }
            break;
        case MODEL_PLATE: {
            if (ocp->n_model_params < 8) { err = "PLATE: 8 params"; return false; }
            int g = (int)D.p[0], nseg = (int)D.p[5];
            if (g < 2 || D.nx != g * g || D.nu != 4 * nseg || D.nr != D.nx || nseg < 1 || nseg > g) { err = "PLATE: sizes inconsistent with g,nseg"; return false; }
            break;
        }
        default: err = "unknown model"; return false;
    }
    const int N = D.N, nx = D.nx, nv = D.nv;
    mm.n = (int64_t)N * nv; mm.m_dyn = (int64_t)N * nx;
    const int64_t n_g = ocp->n_g;
    if (n_g < 0 || (n_g > 0 && (!ocp->g_rowptr || !ocp->g_colind || !ocp->g_val || !ocp->g_lo || !ocp->g_hi))) { err = "bad general rows"; return false; }
    mm.m = mm.m_dyn + n_g;
    if (mm.n > INT32_MAX / 2 || mm.m > INT32_MAX / 2) { err = "OCP too large for int32 indices"; return false; }
    mm.present = true;
    const int64_t n = mm.n, m = mm.m, m_dyn = mm.m_dyn;
    mm.cl.assign(m, 0.0); mm.cu.assign(m, 0.0); mm.g_val.clear();

    // ---- J pattern: run the row enumerators on a dummy interior point ----
    std::vector<double> xd(nx, 0.5), ud(std::max(1, D.nu), 0.5);
    mm.J.nrows = m; mm.J.ncols = n; mm.J.ptr.assign(m + 1, 0);
    mm.J.idx.clear(); mm.J.idx.reserve((size_t)m * 6);
    for (int k = 0; k < N; ++k)
        for (int c = 0; c < nx; ++c) {
            if (k > 0) mm.J.idx.push_back((k - 1) * nv + c);
            auto emit = [&](int col, double) { mm.J.idx.push_back(k * nv + col); };
            model_row(D, c, xd.data(), ud.data(), emit);
            mm.J.ptr[(int64_t)k * nx + c + 1] = (int64_t)mm.J.idx.size();
        }
    // ---- the general linear rows lo <= G y <= hi below the dynamics rows (include/nmpc.h: nmpc_ocp) ----
    for (int64_t g = 0; g < n_g; ++g) {
        const int64_t a = ocp->g_rowptr[g], b = ocp->g_rowptr[g + 1];
        if (g == 0 && a != 0) { err = "g_rowptr[0] != 0"; return false; }
        if (b <= a) { err = "empty general row"; return false; }
        for (int64_t p = a; p < b; ++p) {
            const int32_t col = ocp->g_colind[p];
            if (col < 0 || col >= n || (p > a && col <= ocp->g_colind[p - 1])) { err = "general row: column out of range or not increasing"; return false; }
            mm.J.idx.push_back(col); mm.g_val.push_back(ocp->g_val[p]);
        }
        mm.J.ptr[m_dyn + g + 1] = (int64_t)mm.J.idx.size();
        if (!(ocp->g_lo[g] <= ocp->g_hi[g])) { err = "general row: lo > hi"; return false; }
        mm.cl[m_dyn + g] = ocp->g_lo[g]; mm.cu[m_dyn + g] = ocp->g_hi[g];
    }
    const int64_t nnzJ = mm.J.nnz();
    for (int64_t r = 0; r < m; ++r) {
        if (r < m_dyn && mm.J.ptr[r + 1] - mm.J.ptr[r] > MAX_JROW + 1) { err = "J row too long"; return false; }
        for (int64_t p = mm.J.ptr[r] + 1; p < mm.J.ptr[r + 1]; ++p)
            if (mm.J.idx[p] <= mm.J.idx[p - 1]) { err = "J row not sorted"; return false; }
    }
    // ---- W pattern (stage-block diagonal, lower) ----
    const int hc = hess_count(D);
    mm.W.nrows = n; mm.W.ncols = n; mm.W.ptr.assign(n + 1, 0); mm.W.idx.resize((size_t)N * hc);
    for (int k = 0; k < N; ++k)
        for (int e = 0; e < hc; ++e) {
            int a, b; hess_pos(D, e, &a, &b);
            mm.W.ptr[(int64_t)k * nv + a + 1]++;
            mm.W.idx[(size_t)k * hc + e] = k * nv + b;
        }
    for (int64_t i = 0; i < n; ++i) mm.W.ptr[i + 1] += mm.W.ptr[i];
    // ---- CSC of J ----
    mm.jt_ptr.assign(n + 1, 0);
    for (int64_t p = 0; p < nnzJ; ++p) mm.jt_ptr[mm.J.idx[p] + 1]++;
    for (int64_t i = 0; i < n; ++i) mm.jt_ptr[i + 1] += mm.jt_ptr[i];
    mm.jt_idx.resize(nnzJ); mm.jt_row.resize(nnzJ);
    {
        std::vector<int64_t> pos(mm.jt_ptr.begin(), mm.jt_ptr.end() - 1);
        for (int64_t r = 0; r < m; ++r)
            for (int64_t p = mm.J.ptr[r]; p < mm.J.ptr[r + 1]; ++p) {
                int64_t q = pos[mm.J.idx[p]]++;
                mm.jt_idx[q] = (int32_t)p; mm.jt_row[q] = (int32_t)r;
            }
    }
    // ---- K pattern: for column j, rows i >= j with (J^T J)_ij != 0, plus W, plus diagonal.  Built row-wise:
    //      row i of lower K = { j <= i : exists r with J_ri, J_rj != 0 } u W row i u {i}
    mm.K.nrows = n; mm.K.ncols = n; mm.K.ptr.assign(n + 1, 0); mm.K.idx.clear();
    {
        std::vector<int32_t> mark(n, -1), buf;
        for (int64_t i = 0; i < n; ++i) {
            buf.clear();
            mark[i] = (int32_t)i; buf.push_back((int32_t)i);
            for (int64_t q = mm.jt_ptr[i]; q < mm.jt_ptr[i + 1]; ++q) {
                int64_t r = mm.jt_row[q];
                for (int64_t p = mm.J.ptr[r]; p < mm.J.ptr[r + 1]; ++p) {
                    int32_t j = mm.J.idx[p];
                    if (j <= i && mark[j] != i) { mark[j] = (int32_t)i; buf.push_back(j); }
                }
            }
            for (int64_t p = mm.W.ptr[i]; p < mm.W.ptr[i + 1]; ++p) {
                int32_t j = mm.W.idx[p];
                if (mark[j] != i) { mark[j] = (int32_t)i; buf.push_back(j); }
            }
            std::sort(buf.begin(), buf.end());
            mm.K.idx.insert(mm.K.idx.end(), buf.begin(), buf.end());
            mm.K.ptr[i + 1] = (int64_t)mm.K.idx.size();
        }
    }
    const int64_t nnzK = mm.K.nnz();
    auto kfind = [&](int64_t i, int32_t j) -> int64_t {
        auto b = mm.K.idx.begin() + mm.K.ptr[i], e = mm.K.idx.begin() + mm.K.ptr[i + 1];
        auto it = std::lower_bound(b, e, j);
        return (it != e && *it == j) ? (int64_t)(it - mm.K.idx.begin()) : -1;
    };
    // ---- gather triples, grouped by K entry, increasing J row inside an entry ----
    mm.trip_ptr.assign(nnzK + 1, 0);
    for (int pass = 0; pass < 2; ++pass) {
        std::vector<int64_t> pos;
        if (pass == 1) {
            for (int64_t e = 0; e < nnzK; ++e) mm.trip_ptr[e + 1] += mm.trip_ptr[e];
            pos.assign(mm.trip_ptr.begin(), mm.trip_ptr.end() - 1);
            int64_t nt = mm.trip_ptr[nnzK];
            if (nt > INT32_MAX) { err = "too many gather triples"; return false; }
            mm.trip_a.resize(nt); mm.trip_b.resize(nt); mm.trip_r.resize(nt);
        }
        for (int64_t r = 0; r < m; ++r)
            for (int64_t pa = mm.J.ptr[r]; pa < mm.J.ptr[r + 1]; ++pa)
                for (int64_t pb = mm.J.ptr[r]; pb <= pa; ++pb) {        // col(pa) >= col(pb): lower entry
                    int64_t e = kfind(mm.J.idx[pa], mm.J.idx[pb]);
                    if (pass == 0) mm.trip_ptr[e + 1]++;
                    else { int64_t q = pos[e]++; mm.trip_a[q] = (int32_t)pa; mm.trip_b[q] = (int32_t)pb; mm.trip_r[q] = (int32_t)r; }
                }
    }
    mm.k_w.assign(nnzK, -1); mm.k_diag.assign(nnzK, -1);
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t p = mm.W.ptr[i]; p < mm.W.ptr[i + 1]; ++p) mm.k_w[kfind(i, mm.W.idx[p])] = (int32_t)p;
        mm.k_diag[kfind(i, (int32_t)i)] = (int32_t)i;
    }
    // NOTE: W values are emitted per stage in hess_pos order (k*hc + e); W.idx above is in that order and, because
    // hess_pos is sorted by (a,b), it coincides with the CSR order of W.
    // ---- coordinates for geometric nested dissection ----
    mm.coords.assign((size_t)n * 3, 0); mm.is_input.assign(n, 0);
    for (int k = 0; k < N; ++k)
        for (int a = 0; a < nv; ++a) {
            int64_t v = (int64_t)k * nv + a;
            int32_t* cd = &mm.coords[v * 3];
            cd[0] = k;
            if (a >= nx) {
                mm.is_input[v] = 1;
                if (D.model == MODEL_PLATE) {
                    int g = (int)D.p[0], nseg = (int)D.p[5], h = a - nx, e = h / nseg, sg = h % nseg;
                    int mid = (int)(((2 * sg + 1) * g) / (2 * nseg));
                    if (e == 0) { cd[1] = 0; cd[2] = mid; } else if (e == 1) { cd[1] = g - 1; cd[2] = mid; }
                    else if (e == 2) { cd[1] = mid; cd[2] = 0; } else { cd[1] = mid; cd[2] = g - 1; }
                } else { cd[1] = nx / 2; cd[2] = 0; }
            } else if (D.model == MODEL_PLATE) {
                int g = (int)D.p[0];
                cd[1] = a / g; cd[2] = a % g;
            } else { cd[1] = a; cd[2] = 0; }
        }
    return true;
}


// =============================================================================================================
// Orderings
// =============================================================================================================
struct Graph {                       // symmetric adjacency without self loops
    int64_t n = 0;
    std::vector<int64_t> ptr;
    std::vector<int32_t> adj;
};

static Graph graph_from_lower(const Csr& K) {
    Graph G; G.n = K.nrows;
    const int64_t n = G.n;
    G.ptr.assign(n + 1, 0);
    for (int64_t i = 0; i < n; ++i)
        for (int64_t p = K.ptr[i]; p < K.ptr[i + 1]; ++p) {
            int32_t j = K.idx[p];
            if (j != i) { G.ptr[i + 1]++; G.ptr[j + 1]++; }
        }
    for (int64_t i = 0; i < n; ++i) G.ptr[i + 1] += G.ptr[i];
    G.adj.resize(G.ptr[n]);
    std::vector<int64_t> pos(G.ptr.begin(), G.ptr.end() - 1);
    for (int64_t i = 0; i < n; ++i)
        for (int64_t p = K.ptr[i]; p < K.ptr[i + 1]; ++p) {
            int32_t j = K.idx[p];
            if (j != i) { G.adj[pos[i]++] = j; G.adj[pos[j]++] = (int32_t)i; }
        }
    return G;
}

// Minimum-degree ordering on the subgraph induced by `nodes` (quotient graph with element absorption and the
// approximate external degree of Amestoy-Davis-Duff, PAPER.md ref. [46]); ties -> most recently updated node,
// deterministic.  `local` is scratch of size G.n filled with -1.  Appends the order to `out`.
static void min_degree(const Graph& G, const std::vector<int32_t>& nodes, std::vector<int32_t>& local,
                       std::vector<int32_t>& out) {
    const int32_t nn = (int32_t)nodes.size();
    if (nn == 0) return;
    for (int32_t a = 0; a < nn; ++a) local[nodes[a]] = a;
    std::vector<std::vector<int32_t>> adj(nn), elems(nn), evars(nn);
    for (int32_t a = 0; a < nn; ++a) {
        int32_t v = nodes[a];
        for (int64_t p = G.ptr[v]; p < G.ptr[v + 1]; ++p) { int32_t b = local[G.adj[p]]; if (b >= 0) adj[a].push_back(b); }
    }
    enum : uint8_t { VAR = 0, ELEM = 1, DEAD = 2 };
    std::vector<uint8_t> state(nn, VAR);
    std::vector<int32_t> deg(nn), head(nn + 1, -1), next(nn, -1), prev(nn, -1), mark(nn, -1), w(nn, -1), wstamp(nn, -1);
    auto bucket_insert = [&](int32_t i) { int32_t d = deg[i]; next[i] = head[d]; prev[i] = -1; if (head[d] >= 0) prev[head[d]] = i; head[d] = i; };
    auto bucket_remove = [&](int32_t i) { int32_t d = deg[i]; if (prev[i] >= 0) next[prev[i]] = next[i]; else head[d] = next[i]; if (next[i] >= 0) prev[next[i]] = prev[i]; };
    for (int32_t a = nn - 1; a >= 0; --a) { deg[a] = (int32_t)adj[a].size(); bucket_insert(a); }
    int32_t mindeg = 0, alive = nn;
    std::vector<int32_t> Lp;
    for (int32_t step = 0; step < nn; ++step) {
        while (mindeg < nn && head[mindeg] < 0) ++mindeg;
        const int32_t p = head[mindeg];
        bucket_remove(p);
        out.push_back(nodes[p]);
        // ---- form element p ----
        Lp.clear(); mark[p] = step;
        for (int32_t v : adj[p]) if (state[v] == VAR && mark[v] != step) { mark[v] = step; Lp.push_back(v); }
        for (int32_t e : elems[p]) {
            if (state[e] != ELEM) continue;
            for (int32_t v : evars[e]) if (state[v] == VAR && mark[v] != step && v != p) { mark[v] = step; Lp.push_back(v); }
            state[e] = DEAD; std::vector<int32_t>().swap(evars[e]);
        }
        state[p] = ELEM; --alive;
        std::vector<int32_t>().swap(adj[p]); std::vector<int32_t>().swap(elems[p]);
        // ---- |Le \ Lp| for the elements touching Lp ----
        for (int32_t i : Lp) {
            size_t k = 0;
            for (int32_t e : elems[i]) {
                if (state[e] != ELEM) continue;
                elems[i][k++] = e;
                if (wstamp[e] != step) { wstamp[e] = step; w[e] = (int32_t)evars[e].size(); }
                --w[e];
            }
            elems[i].resize(k);
        }
        // ---- update the variables of Lp ----
        const int32_t lp = (int32_t)Lp.size();
        for (int32_t i : Lp) {
            size_t k = 0;
            for (int32_t v : adj[i]) if (state[v] == VAR && mark[v] != step) adj[i][k++] = v;     // covered by element p
            adj[i].resize(k);
            int64_t d = (int64_t)adj[i].size() + (lp - 1);
            k = 0;
            for (int32_t e : elems[i]) {
                if (w[e] == 0) continue;                    // e is a subset of Lp: absorbed (aggressive absorption)
                elems[i][k++] = e; d += w[e];
            }
            elems[i].resize(k);
            elems[i].push_back(p);
            int64_t cap = std::min<int64_t>(alive - 1, (int64_t)deg[i] + (lp - 1));
            if (d > cap) d = cap;
            if (d < 0) d = 0;
            bucket_remove(i);
            deg[i] = (int32_t)d;
            bucket_insert(i);
            if (deg[i] < mindeg) mindeg = deg[i];
        }
        for (int32_t i : Lp) for (int32_t e : elems[i]) if (e != p && wstamp[e] == step && w[e] == 0 && state[e] == ELEM) { state[e] = DEAD; std::vector<int32_t>().swap(evars[e]); }
        evars[p] = Lp;
    }
    for (int32_t a = 0; a < nn; ++a) local[nodes[a]] = -1;
}

struct NdCtx {
    const Graph* G;
    const int32_t* coords;        // n x 3 or NULL
    const uint8_t* hub;           // n or NULL
    int dims_mask;                // bit d set: dimension d may be cut
    int32_t leaf;
    std::vector<int32_t> side;    // n: scratch, -1 outside the current set; 0 = A, 1 = B, 2 = S
    std::vector<int32_t> local;   // n: scratch for min_degree
    std::vector<int32_t> order;   // output
};

// one-sided vertex separator of the split (side 0 / side 1): returns the nodes of side 0 adjacent to side 1, after
// optionally moving hub nodes of side 1 that touch side 0 into the separator.
static void extract_separator(NdCtx& C, const std::vector<int32_t>& nodes, bool use_hubs, std::vector<int32_t>& S) {
    const Graph& G = *C.G;
    S.clear();
    if (use_hubs && C.hub)
        for (int32_t v : nodes)
            if (C.side[v] == 1 && C.hub[v])
                for (int64_t p = G.ptr[v]; p < G.ptr[v + 1]; ++p)
                    if (C.side[G.adj[p]] == 0) { C.side[v] = 2; S.push_back(v); break; }
    for (int32_t v : nodes)
        if (C.side[v] == 0)
            for (int64_t p = G.ptr[v]; p < G.ptr[v + 1]; ++p)
                if (C.side[G.adj[p]] == 1) { C.side[v] = 2; S.push_back(v); break; }
}

static void nd_recurse(NdCtx& C, std::vector<int32_t>& nodes) {
    const Graph& G = *C.G;
    const int64_t cnt = (int64_t)nodes.size();
    if (cnt == 0) return;
    auto do_leaf = [&]() { min_degree(G, nodes, C.local, C.order); };
    if (cnt <= C.leaf) { do_leaf(); return; }
    // candidate splits: ((dimension, hub rule) -> separator size); keep the best
    struct Cand { int dim; bool hubs; int32_t thr; double cost; };
    Cand best{-1, false, 0, 1e300};
    std::vector<int32_t> S, vals;
    std::vector<int32_t> bfs_level;                // used when no coordinates: "dimension" 0 = BFS level
    const bool have_coords = C.coords != nullptr;
    if (!have_coords) {
        // pseudo-peripheral start: two BFS sweeps inside the current set
        for (int32_t v : nodes) C.side[v] = 0;
        bfs_level.assign(cnt, -1);
        std::vector<int32_t> q; q.reserve(cnt);
        int32_t start = nodes[0];
        for (int sweep = 0; sweep < 3; ++sweep) {
            for (int32_t v : nodes) C.local[v] = -1;
            q.clear(); q.push_back(start); C.local[start] = 0;
            for (size_t h = 0; h < q.size(); ++h) {
                int32_t v = q[h];
                for (int64_t p = G.ptr[v]; p < G.ptr[v + 1]; ++p) {
                    int32_t u = G.adj[p];
                    if (C.side[u] == 0 && C.local[u] < 0) { C.local[u] = C.local[v] + 1; q.push_back(u); }
                }
            }
            start = q.back();
            if ((int64_t)q.size() < cnt) break;     // disconnected: handled below
        }
        int32_t far = 0;
        for (int32_t v : nodes) far = std::max(far, C.local[v]);
        for (int64_t a = 0; a < cnt; ++a) { int32_t l = C.local[nodes[a]]; bfs_level[a] = l < 0 ? far + 1 : l; }   // unreachable -> last level
        for (int32_t v : nodes) { C.local[v] = -1; C.side[v] = -1; }
    }
    auto coord_of = [&](int64_t a, int d) -> int32_t { return have_coords ? C.coords[(int64_t)nodes[a] * 3 + d] : bfs_level[a]; };
    const int ndims = have_coords ? 3 : 1;
    for (int d = 0; d < ndims; ++d) {
        if (have_coords && !((C.dims_mask >> d) & 1)) continue;
        vals.resize(cnt);
        for (int64_t a = 0; a < cnt; ++a) vals[a] = coord_of(a, d);
        std::vector<int32_t> sorted(vals);
        std::nth_element(sorted.begin(), sorted.begin() + cnt / 2, sorted.end());
        int32_t med = sorted[cnt / 2];
        int32_t lo = *std::min_element(vals.begin(), vals.end());
        if (lo == med) {                        // everything below the median is empty: cut above it instead
            int32_t nxt = INT32_MAX;
            for (int32_t v : vals) if (v > med && v < nxt) nxt = v;
            if (nxt == INT32_MAX) continue;     // single coordinate value: cannot cut this dimension
            med = nxt;
        }
        for (int hb = 0; hb < (C.hub ? 2 : 1); ++hb) {
            int64_t na = 0, nb = 0;
            for (int64_t a = 0; a < cnt; ++a) { bool A = vals[a] < med; C.side[nodes[a]] = A ? 0 : 1; (A ? na : nb)++; }
            extract_separator(C, nodes, hb == 1, S);
            int64_t a2 = 0, b2 = 0;
            for (int32_t v : nodes) { if (C.side[v] == 0) ++a2; else if (C.side[v] == 1) ++b2; }
            double imb = (double)std::max(a2, b2) / (double)std::max<int64_t>(1, a2 + b2);
            double cost = (double)S.size() * (1.0 + 2.0 * std::max(0.0, imb - 0.6));
            if (a2 == 0 || b2 == 0) cost = 1e299;
            if (cost < best.cost) best = Cand{d, hb == 1, med, cost};
        }
    }
    for (int32_t v : nodes) C.side[v] = -1;
    if (best.dim < 0 || best.cost >= 1e299) { do_leaf(); return; }
    for (int64_t a = 0; a < cnt; ++a) C.side[nodes[a]] = coord_of(a, best.dim) < best.thr ? 0 : 1;
    extract_separator(C, nodes, best.hubs, S);
    std::vector<int32_t> A, B;
    for (int32_t v : nodes) { if (C.side[v] == 0) A.push_back(v); else if (C.side[v] == 1) B.push_back(v); }
    for (int32_t v : nodes) C.side[v] = -1;
    std::vector<int32_t> Sep(S);
    std::vector<int32_t>().swap(nodes);
    nd_recurse(C, A);
    nd_recurse(C, B);
    std::sort(Sep.begin(), Sep.end());
    for (int32_t v : Sep) C.order.push_back(v);
}

static void order_nd(const Graph& G, const int32_t* coords, const uint8_t* hub, int dims_mask, int32_t leaf,
                     std::vector<int32_t>& perm) {
    NdCtx C;
    C.G = &G; C.coords = coords; C.hub = hub; C.dims_mask = dims_mask; C.leaf = std::max(1, leaf);
    C.side.assign(G.n, -1); C.local.assign(G.n, -1);
    C.order.reserve(G.n);
    std::vector<int32_t> all(G.n);
    std::iota(all.begin(), all.end(), 0);
    nd_recurse(C, all);
    perm = C.order;
}


// =============================================================================================================
// Elimination tree, column counts, supernodes, maps
// =============================================================================================================
struct PermutedLower {                 // B = P K P^T, lower triangle, both CSR (rows) and CSC (columns) + source index
    std::vector<int64_t> rptr, cptr;
    std::vector<int32_t> rcol, crow;
    std::vector<int32_t> csrc;         // K value index of CSC entry
};

static void permute_lower(const Csr& K, const std::vector<int32_t>& iperm, PermutedLower& B) {
    const int64_t n = K.nrows, nnz = K.nnz();
    B.rptr.assign(n + 1, 0); B.cptr.assign(n + 1, 0);
    for (int64_t i = 0; i < n; ++i)
        for (int64_t p = K.ptr[i]; p < K.ptr[i + 1]; ++p) {
            int32_t a = iperm[i], b = iperm[K.idx[p]];
            int32_t r = std::max(a, b), c = std::min(a, b);
            B.rptr[r + 1]++; B.cptr[c + 1]++;
        }
    for (int64_t i = 0; i < n; ++i) { B.rptr[i + 1] += B.rptr[i]; B.cptr[i + 1] += B.cptr[i]; }
    B.rcol.resize(nnz); B.crow.resize(nnz); B.csrc.resize(nnz);
    std::vector<int64_t> rp(B.rptr.begin(), B.rptr.end() - 1), cp(B.cptr.begin(), B.cptr.end() - 1);
    for (int64_t i = 0; i < n; ++i)
        for (int64_t p = K.ptr[i]; p < K.ptr[i + 1]; ++p) {
            int32_t a = iperm[i], b = iperm[K.idx[p]];
            int32_t r = std::max(a, b), c = std::min(a, b);
            B.rcol[rp[r]++] = c;
            int64_t q = cp[c]++; B.crow[q] = r; B.csrc[q] = (int32_t)p;
        }
}

// Liu's elimination-tree algorithm with path compression, from the rows of the lower triangle:
// parent[j] = min{ i > j : L_ij != 0 }.
static void elimination_tree(int64_t n, const PermutedLower& B, std::vector<int32_t>& parent) {
    parent.assign(n, -1);
    std::vector<int32_t> anc(n, -1);
    for (int64_t i = 0; i < n; ++i)
        for (int64_t p = B.rptr[i]; p < B.rptr[i + 1]; ++p) {
            int32_t r = B.rcol[p];
            while (r != -1 && r < i) {
                int32_t nx = anc[r];
                anc[r] = (int32_t)i;
                if (nx == -1) parent[r] = (int32_t)i;
                r = nx;
            }
        }
}

static void postorder(const std::vector<int32_t>& parent, std::vector<int32_t>& post) {
    const int64_t n = (int64_t)parent.size();
    std::vector<int32_t> head(n, -1), next(n, -1);
    for (int64_t j = n - 1; j >= 0; --j) if (parent[j] >= 0) { next[j] = head[parent[j]]; head[parent[j]] = (int32_t)j; }
    post.clear(); post.reserve(n);
    std::vector<int32_t> stack;
    for (int64_t root = 0; root < n; ++root) {
        if (parent[root] >= 0) continue;
        stack.push_back((int32_t)root);
        while (!stack.empty()) {
            int32_t v = stack.back();
            int32_t c = head[v];
            if (c >= 0) { head[v] = next[c]; stack.push_back(c); }
            else { post.push_back(v); stack.pop_back(); }
        }
    }
}

static bool validate_pattern(const nmpc_pattern* P, std::string& err) {
    if (!P || P->n <= 0 || !P->rowptr || !P->colind) { err = "null or empty pattern"; return false; }
    if (P->n > INT32_MAX / 2) { err = "n too large for int32 indices"; return false; }
    if (P->rowptr[0] != 0 || P->rowptr[P->n] != P->nnz) { err = "rowptr[0] != 0 or rowptr[n] != nnz"; return false; }
    if (P->nnz > INT32_MAX) { err = "nnz(K) too large for int32 value indices"; return false; }
    for (int64_t i = 0; i < P->n; ++i) {
        int64_t a = P->rowptr[i], b = P->rowptr[i + 1];
        if (b <= a) { err = "row " + std::to_string(i) + " is empty (diagonal missing)"; return false; }
        for (int64_t p = a; p < b; ++p) {
            int32_t j = P->colind[p];
            if (j < 0 || j > i) { err = "row " + std::to_string(i) + " has an entry above the diagonal or out of range"; return false; }
            if (p > a && j <= P->colind[p - 1]) { err = "row " + std::to_string(i) + " unsorted or duplicate"; return false; }
        }
        if (P->colind[b - 1] != i) { err = "row " + std::to_string(i) + " has no diagonal entry"; return false; }
    }
    return true;
}

nmpc_status analyze_symbolic(const nmpc_pattern* pattern, const nmpc_ocp* ocp, const nmpc_options* opt_in, Symbolic& S, bool augment) {
    auto t0 = std::chrono::steady_clock::now();
    nmpc_options opt;
    if (opt_in) opt = *opt_in; else default_options(&opt);
    if (!build_model_maps(ocp, S.mm, S.error)) return NMPC_E_ARG;
    if (pattern) {
        if (!validate_pattern(pattern, S.error)) return NMPC_E_PATTERN;
        S.K.nrows = S.K.ncols = pattern->n;
        S.K.ptr.assign(pattern->rowptr, pattern->rowptr + pattern->n + 1);
        S.K.idx.assign(pattern->colind, pattern->colind + pattern->nnz);
        if (S.mm.present) {
            // the model's K pattern must be the given pattern (value order of the assembly kernel)
            if (pattern->n != S.mm.n || S.K.ptr != S.mm.K.ptr || S.K.idx != S.mm.K.idx) {
                S.error = "pattern differs from the model's K pattern (pass pattern = NULL to derive it)"; return NMPC_E_PATTERN;
            }
        }
    } else {
        if (!S.mm.present) { S.error = "no pattern and no model"; return NMPC_E_ARG; }
        S.K = S.mm.K;
    }
    const int64_t n = S.K.nrows;
    S.n = n; S.nnzK = S.K.nnz();

    // ---------------- ordering (Eq. 18: P) ----------------
    Graph G = graph_from_lower(S.K);
    int ordering = opt.ordering;
    if (ordering == NMPC_ORDER_AUTO) ordering = (n <= 64) ? NMPC_ORDER_NATURAL : (S.mm.present ? NMPC_ORDER_ND : NMPC_ORDER_AMD);
    S.ordering_used = ordering;
    std::vector<int32_t> perm(n);
    std::iota(perm.begin(), perm.end(), 0);
    if (ordering == NMPC_ORDER_AMD) {
        std::vector<int32_t> local(n, -1), nodes(perm), out; out.reserve(n);
        min_degree(G, nodes, local, out);
        perm = out;
    } else if (ordering == NMPC_ORDER_ND || ordering == NMPC_ORDER_TIME_ND) {
        int32_t leaf = opt.nd_leaf;
        const int32_t* coords = S.mm.present ? S.mm.coords.data() : nullptr;
        const uint8_t* hub = S.mm.present ? S.mm.is_input.data() : nullptr;
        int mask = 7;
        if (ordering == NMPC_ORDER_TIME_ND) { if (!coords) { S.error = "TIME_ND needs a stage-structured OCP"; return NMPC_E_ARG; } mask = 1; }
        if (leaf <= 0) leaf = (ordering == NMPC_ORDER_TIME_ND) ? S.mm.desc.nv : 96;
        order_nd(G, coords, hub, mask, leaf, perm);
    }
    if ((int64_t)perm.size() != n) { S.error = "internal: ordering lost variables"; return NMPC_E_ARG; }

    // ---------------- right-hand-side row (symbolic.h): [K b; b^T 0], the extra variable n ordered last ----------------
    // Its entries take the value indices nnzK .. nnzK + n (the CSR order of the augmented pattern), i.e. the value array
    // of the numeric factorization is [K values | b | 0].  The ordering above was computed on K alone.
    const int64_t nt = n + (augment ? 1 : 0);
    S.aug = augment; S.nt = nt;
    Csr Kaug;
    if (augment) {
        if (S.nnzK + n + 1 > INT32_MAX) { S.error = "nnz(K) too large for int32 value indices"; return NMPC_E_ALLOC; }
        Kaug.nrows = Kaug.ncols = nt;
        Kaug.ptr = S.K.ptr; Kaug.ptr.push_back(S.nnzK + n + 1);
        Kaug.idx = S.K.idx; Kaug.idx.resize(S.nnzK + n + 1);
        std::iota(Kaug.idx.begin() + S.nnzK, Kaug.idx.end(), 0);
        perm.push_back((int32_t)n);
    }
    const Csr& Kf = augment ? Kaug : S.K;
    S.nnzKa = Kf.nnz();

    // ---------------- etree + postorder, then redo on the postordered permutation ----------------
    std::vector<int32_t> iperm(nt);
    PermutedLower B;
    for (int round = 0; round < 2; ++round) {
        for (int64_t i = 0; i < nt; ++i) iperm[perm[i]] = (int32_t)i;
        permute_lower(Kf, iperm, B);
        elimination_tree(nt, B, S.parent);
        if (round == 0) {
            std::vector<int32_t> post, np(nt);
            postorder(S.parent, post);
            for (int64_t k = 0; k < nt; ++k) np[k] = perm[post[k]];
            perm.swap(np);
        }
    }
    if (augment && perm[n] != n) { S.error = "internal: the right-hand-side row is not the last pivot"; return NMPC_E_ARG; }
    S.perm = perm; S.iperm = iperm;
    // rows of B sorted by column (needed nowhere), columns of B: sort each column's rows (keeps diagonal first)
    for (int64_t j = 0; j < nt; ++j) {
        int64_t a = B.cptr[j], b = B.cptr[j + 1];
        std::vector<std::pair<int32_t, int32_t>> tmp(b - a);
        for (int64_t p = a; p < b; ++p) tmp[p - a] = {B.crow[p], B.csrc[p]};
        std::sort(tmp.begin(), tmp.end());
        for (int64_t p = a; p < b; ++p) { B.crow[p] = tmp[p - a].first; B.csrc[p] = tmp[p - a].second; }
    }
    // ---------------- column counts by row-subtree traversal ----------------
    S.colcount.assign(nt, 1);
    {
        std::vector<int32_t> mark(nt, -1);
        for (int64_t i = 0; i < nt; ++i) {
            mark[i] = (int32_t)i;
            for (int64_t p = B.rptr[i]; p < B.rptr[i + 1]; ++p) {
                int32_t k = B.rcol[p];
                while (k != -1 && k < i && mark[k] != i) { S.colcount[k]++; mark[k] = (int32_t)i; k = S.parent[k]; }
            }
        }
    }
    S.flops = 0.0;
    // algorithmic flops of the factorization of K itself (the right-hand-side row is not counted)
    for (int64_t j = 0; j < n; ++j) { const double cc = (double)(S.colcount[j] - (augment ? 1 : 0)); S.flops += cc * cc; }

    // ---------------- maximal supernodes, then relaxed amalgamation ----------------
    struct SN { int32_t start, w, r; int64_t zeros; int32_t parent_col; };
    std::vector<SN> sn;
    for (int64_t j = 0; j < nt; ++j) {
        if (!sn.empty() && S.parent[j - 1] == j && S.colcount[j] == S.colcount[j - 1] - 1) sn.back().w++;
        else sn.push_back(SN{(int32_t)j, 1, S.colcount[j], 0, -1});
    }
    auto panel_nnz = [](int64_t r, int64_t w) { return r * w - w * (w - 1) / 2; };
    {
        // parent column of a supernode = etree parent of its last column
        std::vector<SN> out;            // stack of finished (possibly merged) supernodes in column order
        for (const SN& s0 : sn) {
            SN cur = s0;
            while (!out.empty()) {
                SN& c = out.back();
                int32_t c_last = c.start + c.w - 1;
                if (c.start + c.w != cur.start) break;
                int32_t pc = S.parent[c_last];
                if (pc < cur.start || pc >= cur.start + cur.w) break;      // c is not a child of cur
                int64_t w2 = (int64_t)c.w + cur.w, r2 = (int64_t)c.w + cur.r;
                int64_t z2 = panel_nnz(r2, w2) - (panel_nnz(c.r, c.w) - c.zeros) - (panel_nnz(cur.r, cur.w) - cur.zeros);
                bool merge = (w2 <= (opt.relax_small < 0 ? 8 : opt.relax_small)) || ((double)z2 <= opt.relax_zeros * (double)panel_nnz(r2, w2));
                if (!merge) break;
                cur.start = c.start; cur.w = (int32_t)w2; cur.r = (int32_t)r2; cur.zeros = z2;
                out.pop_back();
            }
            out.push_back(cur);
        }
        sn.swap(out);
    }
    const int32_t ns = (int32_t)sn.size();
    S.ns = ns;
    S.sn_start.resize(ns + 1); S.sn_of_col.resize(nt);
    for (int32_t s = 0; s < ns; ++s) { S.sn_start[s] = sn[s].start; for (int32_t j = 0; j < sn[s].w; ++j) S.sn_of_col[sn[s].start + j] = s; }
    S.sn_start[ns] = (int32_t)nt;

    // ---------------- row structure of every supernode (bottom-up), supernodal tree ----------------
    S.rows_ptr.assign(ns + 1, 0); S.rows.clear();
    S.sn_parent.assign(ns, -1); S.sn_level.assign(ns, 0);
    std::vector<std::vector<int32_t>> children(ns);
    {
        std::vector<int32_t> mark(nt, -1), buf;
        for (int32_t s = 0; s < ns; ++s) {
            const int32_t c0 = S.sn_start[s], c1 = S.sn_start[s + 1];
            buf.clear();
            for (int32_t j = c0; j < c1; ++j) mark[j] = s;
            for (int32_t j = c0; j < c1; ++j)
                for (int64_t p = B.cptr[j]; p < B.cptr[j + 1]; ++p) {
                    int32_t i = B.crow[p];
                    if (i >= c1 && mark[i] != s) { mark[i] = s; buf.push_back(i); }
                }
            for (int32_t c : children[s]) {
                const int32_t wc = S.sn_start[c + 1] - S.sn_start[c];
                for (int64_t p = S.rows_ptr[c] + wc; p < S.rows_ptr[c + 1]; ++p) {
                    int32_t i = S.rows[p];
                    if (i >= c1 && mark[i] != s) { mark[i] = s; buf.push_back(i); }
                }
            }
            std::sort(buf.begin(), buf.end());
            for (int32_t j = c0; j < c1; ++j) S.rows.push_back(j);
            S.rows.insert(S.rows.end(), buf.begin(), buf.end());
            S.rows_ptr[s + 1] = (int64_t)S.rows.size();
            if (!buf.empty()) { int32_t p = S.sn_of_col[buf[0]]; S.sn_parent[s] = p; children[p].push_back(s); }
        }
    }
    S.child_ptr.assign(ns + 1, 0); S.child_idx.clear();
    for (int32_t s = 0; s < ns; ++s) {
        for (int32_t c : children[s]) { S.child_idx.push_back(c); S.sn_level[s] = std::max(S.sn_level[s], S.sn_level[c] + 1); }
        S.child_ptr[s + 1] = (int32_t)S.child_idx.size();
    }
    S.nlevels = 0;
    for (int32_t s = 0; s < ns; ++s) S.nlevels = std::max(S.nlevels, S.sn_level[s] + 1);
    S.lvl_ptr.assign(S.nlevels + 1, 0);
    for (int32_t s = 0; s < ns; ++s) S.lvl_ptr[S.sn_level[s] + 1]++;
    for (int32_t l = 0; l < S.nlevels; ++l) S.lvl_ptr[l + 1] += S.lvl_ptr[l];
    S.lvl_sn.resize(ns);
    {
        std::vector<int32_t> pos(S.lvl_ptr.begin(), S.lvl_ptr.end() - 1);
        for (int32_t s = 0; s < ns; ++s) S.lvl_sn[pos[S.sn_level[s]]++] = s;
    }
    // ---------------- storage offsets, relative indices, K scatter map ----------------
    S.panel_ptr.assign(ns + 1, 0); S.upd_ptr.assign(ns + 1, 0); S.rel_ptr.assign(ns + 1, 0);
    S.nnzL = 0; S.max_front = 0; S.max_width = 0;
    for (int32_t s = 0; s < ns; ++s) {
        int64_t r = S.rows_ptr[s + 1] - S.rows_ptr[s], w = S.sn_start[s + 1] - S.sn_start[s];
        S.panel_ptr[s + 1] = S.panel_ptr[s] + panel_ld(r) * w;
        S.upd_ptr[s + 1] = S.upd_ptr[s] + (r - w) * (r - w);
        S.rel_ptr[s + 1] = S.rel_ptr[s] + (r - w);
        S.nnzL += panel_nnz(r, w);
        S.max_front = std::max<int32_t>(S.max_front, (int32_t)r);
        S.max_width = std::max<int32_t>(S.max_width, (int32_t)w);
        if (panel_ld(r) * w > INT32_MAX || r > 65535) { S.error = "front too large (panel offsets are int32, front rows uint16)"; return NMPC_E_ALLOC; }
    }
    S.rel.assign(S.rel_ptr[ns], 0);
    for (int32_t s = 0; s < ns; ++s) {
        int32_t p = S.sn_parent[s];
        if (p < 0) continue;
        const int64_t w = S.sn_start[s + 1] - S.sn_start[s];
        int64_t a = S.rows_ptr[s] + w, ae = S.rows_ptr[s + 1], b = S.rows_ptr[p], be = S.rows_ptr[p + 1], q = S.rel_ptr[s];
        for (; a < ae; ++a, ++q) {
            while (b < be && S.rows[b] < S.rows[a]) ++b;
            if (b == be || S.rows[b] != S.rows[a]) { S.error = "internal: child rows not nested in parent"; return NMPC_E_ARG; }
            S.rel[q] = (int32_t)(b - S.rows_ptr[p]);
        }
    }
    S.kent_ptr.assign(ns + 1, 0); S.kent_src.resize(S.nnzKa); S.kent_dst.resize(S.nnzKa);
    {
        int64_t q = 0;
        for (int32_t s = 0; s < ns; ++s) {
            const int32_t c0 = S.sn_start[s], c1 = S.sn_start[s + 1];
            const int64_t r = S.rows_ptr[s + 1] - S.rows_ptr[s], ld = panel_ld(r);
            const int32_t* rw = &S.rows[S.rows_ptr[s]];
            for (int32_t j = c0; j < c1; ++j) {
                int64_t pos = 0;
                for (int64_t p = B.cptr[j]; p < B.cptr[j + 1]; ++p) {          // rows increasing
                    int32_t i = B.crow[p];
                    while (pos < r && rw[pos] < i) ++pos;
                    if (pos == r || rw[pos] != i) { S.error = "internal: K entry outside the supernode structure"; return NMPC_E_ARG; }
                    S.kent_src[q] = B.csrc[p];
                    S.kent_dst[q] = (int32_t)(pos + (int64_t)(j - c0) * ld);
                    ++q;
                }
            }
            S.kent_ptr[s + 1] = q;
        }
    }
    // ---------------- what the C-ABI reports: the structure of the factor of K alone ----------------
    if (augment) {
        S.v_sn_start = S.sn_start; S.v_sn_start[ns] = (int32_t)n;
        S.v_rows_ptr.assign(ns + 1, 0); S.v_rows.clear();
        S.v_nnzL = 0; S.v_panel_doubles = 0; S.v_update_doubles = 0; S.v_max_front = 0; S.v_max_width = 0;
        for (int32_t s = 0; s < ns; ++s) {
            for (int64_t p = S.rows_ptr[s]; p < S.rows_ptr[s + 1]; ++p) if (S.rows[p] != n) S.v_rows.push_back(S.rows[p]);
            S.v_rows_ptr[s + 1] = (int64_t)S.v_rows.size();
            const int64_t r = S.v_rows_ptr[s + 1] - S.v_rows_ptr[s], w = S.v_sn_start[s + 1] - S.v_sn_start[s];
            S.v_nnzL += panel_nnz(r, w); S.v_panel_doubles += panel_ld(r) * w; S.v_update_doubles += (r - w) * (r - w);
            S.v_max_front = std::max<int32_t>(S.v_max_front, (int32_t)r); S.v_max_width = std::max<int32_t>(S.v_max_width, (int32_t)w);
        }
    }
    S.analyze_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return NMPC_OK;
}

}  // namespace nmpc

// =============================================================================================================
// C-ABI: host-only symbolic entry points
// =============================================================================================================
struct nmpc_symbolic_s { nmpc::Symbolic S; };

extern "C" {

void nmpc_default_options(nmpc_options* out) { if (out) nmpc::default_options(out); }

nmpc_status nmpc_symbolic_analyze(const nmpc_pattern* pattern, const nmpc_ocp* ocp, const nmpc_options* opt, nmpc_symbolic* out) {
    if (!out) return NMPC_E_ARG;
    *out = nullptr;
    nmpc_symbolic_s* h = new (std::nothrow) nmpc_symbolic_s();
    if (!h) return NMPC_E_ALLOC;
    nmpc_status st;
    try { st = nmpc::analyze_symbolic(pattern, ocp, opt, h->S, opt && opt->fuse_rhs > 0); }   // host-only analysis: the right-hand-side row on request only
    catch (const std::bad_alloc&) { st = NMPC_E_ALLOC; }
    catch (...) { st = NMPC_E_ARG; }
    if (st != NMPC_OK) { delete h; return st; }
    *out = h;
    return NMPC_OK;
}

void nmpc_fill_info(const nmpc::Symbolic& S, nmpc_sym_info* o) {
    o->n = S.n; o->nnz_K = S.nnzK; o->nnz_L = S.aug ? S.v_nnzL : S.nnzL;
    o->panel_doubles = S.aug ? S.v_panel_doubles : S.panel_ptr.back(); o->update_doubles = S.aug ? S.v_update_doubles : S.upd_ptr.back();
    o->flops = S.flops; o->nsuper = S.ns; o->nlevels = S.nlevels;
    o->max_front = S.aug ? S.v_max_front : S.max_front; o->max_width = S.aug ? S.v_max_width : S.max_width;
    o->n_large_fronts = 0; o->ordering_used = S.ordering_used; o->analyze_ms = S.analyze_ms;
    // with the right-hand-side row (options.fuse_rhs) the arrays describe the factor of K alone: that row is left out (the
    // last supernode may then be empty when K's own structure ends in a separate root); etree_parent of a root of K's
    // forest is n
    o->perm = S.perm.data();
    o->super_start = S.aug ? S.v_sn_start.data() : S.sn_start.data();
    o->rows_ptr = S.aug ? S.v_rows_ptr.data() : S.rows_ptr.data(); o->rows = S.aug ? S.v_rows.data() : S.rows.data();
    o->super_parent = S.sn_parent.data(); o->super_level = S.sn_level.data(); o->etree_parent = S.parent.data();
    o->fused_rhs = S.aug ? 1 : 0;
}

nmpc_status nmpc_symbolic_info(nmpc_symbolic sym, nmpc_sym_info* out) {
    if (!sym || !out) return NMPC_E_ARG;
    nmpc_fill_info(sym->S, out);
    return NMPC_OK;
}

static nmpc_status copy_pattern(const nmpc::Csr& P, int64_t* nnz, int64_t* rowptr, int32_t* colind) {
    if (!nnz) return NMPC_E_ARG;
    *nnz = P.nnz();
    if (rowptr) std::memcpy(rowptr, P.ptr.data(), sizeof(int64_t) * P.ptr.size());
    if (colind) std::memcpy(colind, P.idx.data(), sizeof(int32_t) * P.idx.size());
    return NMPC_OK;
}
nmpc_status nmpc_copy_pattern_internal(const nmpc::Csr& P, int64_t* nnz, int64_t* rowptr, int32_t* colind) { return copy_pattern(P, nnz, rowptr, colind); }

nmpc_status nmpc_symbolic_pattern(nmpc_symbolic sym, int64_t* nnz, int64_t* rowptr, int32_t* colind) {
    if (!sym) return NMPC_E_ARG;
    return copy_pattern(sym->S.K, nnz, rowptr, colind);
}

nmpc_status nmpc_symbolic_kmap(nmpc_symbolic sym, int32_t* super_of_entry, int64_t* panel_offset) {
    if (!sym || !super_of_entry || !panel_offset) return NMPC_E_ARG;
    const nmpc::Symbolic& S = sym->S;
    int64_t voff = 0;                                    // panel offsets in the layout nmpc_get_info / nmpc_get_factor report
    for (int32_t s = 0; s < S.ns; ++s) {
        const int64_t ld = nmpc::panel_ld(S.rows_ptr[s + 1] - S.rows_ptr[s]);
        const int64_t ldv = S.aug ? nmpc::panel_ld(S.v_rows_ptr[s + 1] - S.v_rows_ptr[s]) : ld;
        for (int64_t q = S.kent_ptr[s]; q < S.kent_ptr[s + 1]; ++q) {
            if (S.kent_src[q] >= S.nnzK) continue;       // entries of the right-hand-side row
            super_of_entry[S.kent_src[q]] = s;
            panel_offset[S.kent_src[q]] = S.aug ? voff + S.kent_dst[q] % ld + (S.kent_dst[q] / ld) * ldv : S.panel_ptr[s] + S.kent_dst[q];
        }
        voff += ldv * ((S.aug ? S.v_sn_start[s + 1] : S.sn_start[s + 1]) - S.sn_start[s]);
    }
    return NMPC_OK;
}

void nmpc_symbolic_destroy(nmpc_symbolic sym) { delete sym; }

}  // extern "C"
