// api.cu -- the C-ABI of include/nmpc.h: handle life cycle, task lists of the persistent factor / solve kernels, and the
// host side of Algorithm 2 (LiftedIPM) / Algorithm 1 lines 9-11.
// Every numeric step runs in the kernels of factor.cu / ipm.cu; the host only sequences launches and takes the
// scalar decisions (barrier update, inertia schedule, termination) from a handful of reduced scalars.
#include <algorithm>
#include <chrono>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <thread>
#include <vector>

#include "device.h"
#include "symbolic.h"

using namespace nmpc;

extern "C" void nmpc_fill_info(const nmpc::Symbolic& S, nmpc_sym_info* o);
extern "C" nmpc_status nmpc_copy_pattern_internal(const nmpc::Csr& P, int64_t* nnz, int64_t* rowptr, int32_t* colind);

namespace {

}  // namespace

struct nmpc_handle_s {
    Symbolic S;
    nmpc_options opt;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    int dev = 0;                       // the device that was current in nmpc_analyze; every entry point re-selects it
    DevSym D;
    DevModel M;
    IpmVectors V{};
    std::vector<void*> allocs;
    DagPlan F;
    uint32_t epoch_f = 0, epoch_sf = 0, epoch_sb = 0, epoch_limit = 1u << 16;   // call numbers of the epoch-valued completion flags:
                                       // factorization, forward half and backward half of the solves
    bool rhs_row_valid = false;        // the factor holds v = L^-1 P b of the right-hand side a fused solve is asked for
    int n_big_fronts = 0;
    double* d_Kval = nullptr;          // values last factored (pattern order)
    double* d_x = nullptr;             // permuted right-hand side / solution
    int64_t* d_full_ptr = nullptr; int32_t* d_full_idx = nullptr; int32_t* d_full_src = nullptr;   // symmetric CSR of K
    double* d_uinit = nullptr;
    double* h_pinned = nullptr;        // pinned host scratch: [0..15] scalars, [16] flag, staging for host-buffer calls
    size_t pinned_doubles = 0;
    bool factored = false, have_state = false, has_model = false;
    double eta_cur = 0.0;
    int64_t launches = 0;
    int nmult = 0;
    std::string err;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    std::vector<cudaEvent_t> it_ev;    // per-iteration events of traced solves (created on first use)
    double* d_par = nullptr;           // device {mu, tau, (uint32) factor call number, then (forward, backward) call numbers per solve}: read by the graph's kernels
    cudaGraphExec_t iter_graph = nullptr;   // one IPM iteration (S6-S10 + the next S2), see capture_iteration_graph
    bool graph_failed = false;
};

namespace {

// Every extern "C" entry point that touches the device runs on the handle's device (the one current in nmpc_analyze) and
// restores the caller's current device on return: handles of several devices can be driven from one host thread.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const nmpc_handle_s* h) {
        if (h && cudaGetDevice(&prev) == cudaSuccess && prev != h->dev) cudaSetDevice(h->dev); else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

thread_local std::string g_create_error;   // message of the last failed nmpc_analyze on this thread: nmpc_last_error(NULL)

#define CK(call)                                                                                      \
    do {                                                                                              \
        cudaError_t e__ = (call);                                                                     \
        if (e__ != cudaSuccess) {                                                                     \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e__);                             \
            return NMPC_E_CUDA;                                                                       \
        }                                                                                             \
    } while (0)

template <class T>
nmpc_status upload(nmpc_handle_s* h, const std::vector<T>& v, const T** out) {
    T* d = nullptr;
    size_t bytes = std::max<size_t>(1, v.size()) * sizeof(T);
    if (cudaMalloc((void**)&d, bytes) != cudaSuccess) { h->err = "cudaMalloc failed (" + std::to_string(bytes) + " B)"; cudaGetLastError(); return NMPC_E_ALLOC; }
    h->allocs.push_back(d);
    if (!v.empty()) CK(cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, h->stream));
    *out = d;
    return NMPC_OK;
}

template <class T>
nmpc_status dalloc(nmpc_handle_s* h, size_t count, T** out, bool zero = true) {
    T* d = nullptr;
    size_t bytes = std::max<size_t>(1, count) * sizeof(T);
    if (cudaMalloc((void**)&d, bytes) != cudaSuccess) { h->err = "cudaMalloc failed (" + std::to_string(bytes) + " B)"; cudaGetLastError(); return NMPC_E_ALLOC; }
    h->allocs.push_back(d);
    if (zero) CK(cudaMemsetAsync(d, 0, bytes, h->stream));
    *out = d;
    return NMPC_OK;
}

#define TRY(x) do { nmpc_status s__ = (x); if (s__ != NMPC_OK) return s__; } while (0)

// ---- task list of the persistent factorization kernel + level lists of the solves ----
nmpc_status build_plan(nmpc_handle_s* h, int small_max_r, int ctas_per_sm, size_t smem_bytes, int solve_ctas_per_sm,
                       size_t solve_smem, int num_sms) {
    const Symbolic& S = h->S;
    const int ns = S.ns;
    auto R = [&](int s) { return (int)(S.rows_ptr[s + 1] - S.rows_ptr[s]); };
    auto W = [&](int s) { return S.sn_start[s + 1] - S.sn_start[s]; };
    std::vector<int32_t> cls(ns), tbase(ns, 0), bbase(ns, 0), target(ns, 1), target_f(ns, 1), target_b(ns, 1), nbp(ns, 0), nbt(ns, 0);
    int64_t slots = 0, bslots = 0;
    h->n_big_fronts = 0;
    for (int s = 0; s < ns; ++s) {
        cls[s] = R(s) > small_max_r;
        if (!cls[s]) continue;
        h->n_big_fronts++;
        nbp[s] = tile_nbp(W(s)); nbt[s] = nbp[s] + tile_nbu(W(s), R(s));
        tbase[s] = (int32_t)slots;
        slots += (int64_t)nbp[s] * nbt[s] + 1 + nbt[s];          // tile flags, one spare, row-progress words (factor.cu)
        target[s] = nbt[s] * (nbt[s] + 1) / 2;
        bbase[s] = (int32_t)bslots; bslots += nbp[s];
        target_f[s] = nbt[s]; target_b[s] = 1;             // backward: the chain task finishes the supernode
        if (slots > INT32_MAX / 2) { h->err = "too many tiles"; return NMPC_E_ALLOC; }
    }
    // K scatter map per front class: small = packed lower offset; tiled = tile-local offset, entries sorted by tile slot
    std::vector<int32_t> ksrc(S.kent_src), kdst(S.kent_dst);
    std::vector<int64_t> tile_kptr((size_t)slots + 1, 0);
    for (int s = 0; s < ns; ++s) {
        const int r = R(s), w = W(s), ld = ld_even(r);
        const int64_t q0 = S.kent_ptr[s], q1 = S.kent_ptr[s + 1];
        if (!cls[s]) {
            for (int64_t q = q0; q < q1; ++q) {
                const int j = S.kent_dst[q] / ld, i = S.kent_dst[q] - j * ld;
                kdst[q] = j * r - (j * (j - 1)) / 2 + (i - j);
            }
            continue;
        }
        std::vector<int32_t> bof(r);                     // block of every front row
        for (int k = 0, i = 0; k < nbt[s]; ++k) { const int e = tile_bound(k + 1, w, r, nbp[s]); for (; i < e; ++i) bof[i] = k; }
        std::vector<std::pair<int64_t, int64_t>> key((size_t)(q1 - q0));   // (slot, q)
        for (int64_t q = q0; q < q1; ++q) {
            const int j = S.kent_dst[q] / ld, i = S.kent_dst[q] - j * ld;
            key[q - q0] = {(int64_t)bof[j] * nbt[s] + bof[i], q};
        }
        std::sort(key.begin(), key.end());
        const int64_t nslot = (int64_t)nbp[s] * nbt[s];
        std::vector<int64_t> cnt((size_t)nslot + 1, 0);
        for (int64_t e = 0; e < q1 - q0; ++e) {
            const int64_t q = key[e].second;
            const int j = S.kent_dst[q] / ld, i = S.kent_dst[q] - j * ld;
            const int I = bof[i], J = bof[j];
            ksrc[q0 + e] = S.kent_src[q];
            kdst[q0 + e] = (i - tile_bound(I, w, r, nbp[s])) + (j - tile_bound(J, w, r, nbp[s])) * 66;
            cnt[key[e].first + 1]++;
        }
        for (int64_t k = 0; k <= nslot; ++k) { if (k) cnt[k] += cnt[k - 1]; tile_kptr[tbase[s] + k] = q0 + cnt[k]; }
    }
    // block boundaries of every child of a tiled parent inside that parent's rows
    std::vector<int64_t> cb_ptr(ns, -1);
    std::vector<int32_t> cbnd;
    for (int c = 0; c < ns; ++c) {
        const int p = S.sn_parent[c];
        if (p < 0 || !cls[p]) continue;
        cb_ptr[c] = (int64_t)cbnd.size();
        const int32_t* rel = S.rel.data() + S.rel_ptr[c];
        const int mc = (int)(S.rel_ptr[c + 1] - S.rel_ptr[c]);
        for (int k = 0; k <= nbt[p]; ++k)
            cbnd.push_back((int32_t)(std::lower_bound(rel, rel + mc, tile_bound(k, W(p), R(p), nbp[p])) - rel));
    }
    // task order: descending upward rank (longest remaining path in micro-seconds of a cost model calibrated on the per-task
    // timelines of profiles/: a block column of a tiled front costs ~30 us on the chain POTRF -> TRSM -> GEMM tail -> POTRF, a
    // tiled front ~45 us of assembly / flag hops on top, and its tile GEMMs run at ~100 GFLOP/s per CTA on the whole machine);
    // children rank above their parent, tile (I,k) above tile (I,J) for k < J -> the order is topological
    const double STEP_US = 30.0, FRONT_US = 45.0, MACHINE_FLOPS_PER_US = 100e3 * (double)num_sms * ctas_per_sm;
    auto upd_flops = [&](int s) {                        // update (Schur complement) tiles: (r-w)^2 w
        const double m = R(s) - W(s); return m * m * W(s);
    };
    auto panel_flops = [&](int s) {                      // panel tiles
        const double r = R(s), m = R(s) - W(s); return (r * r * r - m * m * m) / 3.0 - m * m * W(s);
    };
    auto front_time = [&](int s) {
        if (!cls[s]) { const double r = R(s), m = R(s) - W(s); return 2.0 + (r * r * r - m * m * m) / 3.0 * 2.0 / 50e3; }   // ~50 GFLOP/s per CTA
        return FRONT_US + nbp[s] * STEP_US + (panel_flops(s) + upd_flops(s)) / MACHINE_FLOPS_PER_US;
    };
    std::vector<double> rank_end(ns, 0.0);
    for (int s = ns - 1; s >= 0; --s) {                  // parents have larger indices (postorder)
        const int p = S.sn_parent[s];
        rank_end[s] = p < 0 ? 0.0 : rank_end[p] + front_time(p);
    }
    struct TK { double rank; int32_t lvl, type, s, I, J; };
    std::vector<TK> tk;
    for (int s = 0; s < ns; ++s) {
        if (!cls[s]) { tk.push_back(TK{rank_end[s] + front_time(s), S.sn_level[s], 0, s, 0, 0}); continue; }
        const double tail = upd_flops(s) / MACHINE_FLOPS_PER_US;
        for (int J = 0; J < nbt[s]; ++J)
            for (int I = J; I < nbt[s]; ++I)
                tk.push_back(TK{rank_end[s] + (J < nbp[s] ? tail + (nbp[s] - J) * STEP_US : 0.0), S.sn_level[s], 1, s, I, J});
    }
    std::stable_sort(tk.begin(), tk.end(), [](const TK& a, const TK& b) {
        if (a.rank != b.rank) return a.rank > b.rank;
        if (a.lvl != b.lvl) return a.lvl < b.lvl;
        if (a.J != b.J) return a.J < b.J;
        if (a.s != b.s) return a.s < b.s;
        return a.I < b.I;
    });
    std::vector<int4> tasks(tk.size());
    for (size_t t = 0; t < tk.size(); ++t) tasks[t] = make_int4(tk[t].type, tk[t].s, tk[t].I, tk[t].J);

    // solve tasks: forward in descending rank (children before parents, block rows in order); backward top-down in the order
    // of an estimated start time (see below)
    struct SK { double rank; int32_t lvl, type, s, I; };
    std::vector<SK> sk;
    {
        auto solve_time = [&](int s) { return cls[s] ? 2.0 + 4.0 * nbp[s] : 3.0; };
        std::vector<double> rend(ns, 0.0);
        for (int s = ns - 1; s >= 0; --s) { const int p = S.sn_parent[s]; rend[s] = p < 0 ? 0.0 : rend[p] + solve_time(p); }
        for (int s = 0; s < ns; ++s) {
            if (!cls[s]) { sk.push_back(SK{rend[s] + solve_time(s), S.sn_level[s], 0, s, 0}); continue; }
            for (int I = 0; I < nbt[s]; ++I)
                sk.push_back(SK{rend[s] + 1.0 + (I < nbp[s] ? 4.0 * (nbp[s] - I) + 1.0 : 0.0), S.sn_level[s], 1, s, I});
        }
        std::stable_sort(sk.begin(), sk.end(), [](const SK& a, const SK& b) {
            if (a.rank != b.rank) return a.rank > b.rank;
            if (a.lvl != b.lvl) return a.lvl < b.lvl;
            if (a.s != b.s) return a.s < b.s;
            return a.I < b.I;
        });
    }
    std::vector<int4> stasks;
    stasks.reserve(2 * sk.size());
    for (const SK& t : sk) stasks.push_back(make_int4(t.type, t.s, t.I, 0));
    const int32_t n_sfwd = (int32_t)stasks.size();
    // Backward.  CTAs claim tasks in list order and WAIT for the dependencies of what they claimed, so the list must follow the
    // time at which tasks become runnable, or the CTAs fill up with waiting tasks while runnable ones queue behind them.  Every
    // item gets an estimated start time from the dependencies it really has (calibrated on the task timelines under profiles/:
    // ~6 us per block column of a chain, ~8 us chain prologue, ~12 us for a chunk task, ~4 us per small supernode):
    //   chunk task (s, J, c): when the latest piece of x its rows touch is published (block k of a tiled ancestor's chain, or
    //                         a small ancestor as a whole);
    //   chain of s (+ its helper sums, contiguous, in the order the chain needs them): when its last chunk task is done;
    //   small supernode: when its parent is done.
    // Estimates increase strictly along every dependency except chain -> helper, so the sorted list is topological up to that
    // one: the chain waits for helpers that come AFTER it, which is safe for any grid >= 2 -- the helpers between the chain and the
    // one it waits for depend only on blocks the chain has already published, so the other CTAs always get to it.
    std::vector<int64_t> pbase(ns, 0);
    int64_t part_doubles = 0;
    std::vector<int32_t> cbase(ns, 0);
    std::vector<int64_t> cdep_ptr(1, 0);
    std::vector<uint32_t> cdep;
    {
        for (int s = 0; s < ns; ++s) {                   // what every chunk of ancestors' rows has to wait for
            cbase[s] = (int32_t)(cdep_ptr.size() - 1);
            if (!cls[s]) continue;
            const int nchunk = (nbt[s] - nbp[s] + BWD_CH - 1) / BWD_CH;
            pbase[s] = part_doubles; part_doubles += (int64_t)nchunk * W(s);
            const int32_t* rw = &S.rows[S.rows_ptr[s]];
            for (int c = 0; c < nchunk; ++c) {
                const int i0 = tile_bound(nbp[s] + c * BWD_CH, W(s), R(s), nbp[s]);
                const int i1 = tile_bound(std::min(nbt[s], nbp[s] + (c + 1) * BWD_CH), W(s), R(s), nbp[s]);
                const size_t first = cdep.size();
                for (int i = i0; i < i1; ++i) {
                    const int a = S.sn_of_col[rw[i]];
                    // word offsets relative to F.sync (layout below): sol_done_b at 3 + 2 ns, blk_b at 3 + 3 ns + slots + bslots
                    const uint32_t word = cls[a] ? (uint32_t)(3 + 3 * (int64_t)ns + slots + bslots + bbase[a] + (rw[i] - S.sn_start[a]) / TILE)
                                                 : (uint32_t)(3 + 2 * (int64_t)ns + a);
                    if (cdep.size() == first || cdep.back() != word) cdep.push_back(word);   // rows increase: equal words are adjacent
                }
                cdep_ptr.push_back((int64_t)cdep.size());
            }
        }
        const double HOP_US = 6.0, PRO_US = 8.0, UPD_US = 12.0, SMALL_US = 4.0;
        std::vector<double> start(ns, 0.0), fin(ns, 0.0);
        auto published = [&](int g) {                    // when x at pivot position g is available to other CTAs
            const int a = S.sn_of_col[g];
            return cls[a] ? start[a] + PRO_US + HOP_US * (nbp[a] - (g - S.sn_start[a]) / TILE) : fin[a];
        };
        struct Item { double key; int32_t kind, s, I; };  // kind 0 small supernode, 1 chain + helpers of s, 2 chunk task
        std::vector<Item> items;
        for (int s = ns - 1; s >= 0; --s) {              // parents have larger indices (postorder)
            const int p = S.sn_parent[s];
            if (!cls[s]) {
                start[s] = p < 0 ? 0.0 : fin[p];
                fin[s] = start[s] + SMALL_US + 0.05 * W(s);
                items.push_back(Item{start[s], 0, s, 0});
                continue;
            }
            const int nchunk = (nbt[s] - nbp[s] + BWD_CH - 1) / BWD_CH;
            const int32_t* rw = &S.rows[S.rows_ptr[s]];
            double last = 0.0;
            for (int c = 0; c < nchunk; ++c) {
                const int i0 = tile_bound(nbp[s] + c * BWD_CH, W(s), R(s), nbp[s]);
                const int i1 = tile_bound(std::min(nbt[s], nbp[s] + (c + 1) * BWD_CH), W(s), R(s), nbp[s]);
                double key = 0.0;
                for (int i = i0; i < i1; ++i) key = std::max(key, published(rw[i]));
                last = std::max(last, key);
                for (int J = nbp[s] - 1; J >= 0; --J) items.push_back(Item{key + 1e-4 * (nbp[s] - 1 - J), 2, s, J | (c << 16)});
            }
            start[s] = nchunk > 0 ? last + UPD_US : 0.0;
            fin[s] = start[s] + PRO_US + HOP_US * nbp[s];
            items.push_back(Item{start[s], 1, s, 0});
        }
        std::stable_sort(items.begin(), items.end(), [](const Item& a, const Item& b) { return a.key < b.key; });
        for (const Item& it : items) {
            if (it.kind == 0) stasks.push_back(make_int4(0, it.s, 0, 1));
            else if (it.kind == 2) stasks.push_back(make_int4(2, it.s, it.I, 1));
            else {
                stasks.push_back(make_int4(3, it.s, 0, 1));
                for (int J = nbp[it.s] - 4; J >= 0; --J) stasks.push_back(make_int4(1, it.s, J, 1));
            }
        }
    }

    DagPlan& F = h->F;
    const int64_t* tl = nullptr; const int4* t4 = nullptr;
    TRY(upload(h, tasks, &t4)); F.ftasks = t4; F.n_ftasks = (int32_t)tasks.size();
    TRY(upload(h, stasks, &t4)); F.stasks = t4; F.n_stasks = (int32_t)stasks.size(); F.n_sfwd = n_sfwd;
    TRY(upload(h, cls, &F.cls)); TRY(upload(h, tbase, &F.tbase)); TRY(upload(h, bbase, &F.bbase));
    TRY(upload(h, target, &F.target)); TRY(upload(h, target_f, &F.target_f)); TRY(upload(h, target_b, &F.target_b));
    TRY(upload(h, tile_kptr, &tl)); F.tile_kptr = tl;
    TRY(upload(h, cb_ptr, &tl)); F.cb_ptr = tl;
    TRY(upload(h, cbnd, &F.cbnd));
    TRY(upload(h, S.sn_parent, &F.sn_parent));
    TRY(upload(h, pbase, &tl)); F.pbase = tl;
    TRY(upload(h, cbase, &F.cbase)); TRY(upload(h, cdep_ptr, &tl)); F.cdep_ptr = tl;
    { const uint32_t* tu = nullptr; TRY(upload(h, cdep, &tu)); F.cdep = tu; }
    TRY(dalloc(h, (size_t)part_doubles, &F.bpart, false)); TRY(dalloc(h, (size_t)S.nt, &F.bsum, false));
    TRY(upload(h, ksrc, &h->D.kent_src)); TRY(upload(h, kdst, &h->D.kent_dst));
    F.sync_words = 3 + 3 * (int64_t)ns + slots + 5 * bslots;
    TRY(dalloc(h, (size_t)F.sync_words, &F.sync));
    F.fac_done = F.sync + 3; F.sol_done_f = F.fac_done + ns; F.sol_done_b = F.sol_done_f + ns;
    F.tile_done = F.sol_done_b + ns; F.blk_f = F.tile_done + slots; F.blk_b = F.blk_f + bslots; F.blk_u = F.blk_b + bslots; F.blk_s = F.blk_u + bslots; F.sub_done = F.blk_s + bslots;

#ifdef NMPC_TRACE_BUILD                                      // measurement build: per-task timestamps (nmpc_get_task_trace, include/nmpc_aids.h)
    TRY(dalloc(h, (size_t)F.n_ftasks * 8, &F.ftrace)); TRY(dalloc(h, (size_t)F.n_stasks * 8, &F.strace));
#endif
    F.small_max_r = small_max_r;
    F.fsmem = smem_bytes; F.ssmem = solve_smem;
    F.fgrid = (int32_t)std::max<int64_t>(1, std::min<int64_t>((int64_t)tasks.size(), (int64_t)num_sms * ctas_per_sm));
    F.sgrid = (int32_t)std::max<int64_t>(1, std::min<int64_t>((int64_t)stasks.size(), (int64_t)num_sms * solve_ctas_per_sm));
    if (h->opt.grid_limit > 0) { F.fgrid = std::min(F.fgrid, h->opt.grid_limit); F.sgrid = std::min(F.sgrid, std::max(2, h->opt.grid_limit)); }
    if (h->n_big_fronts > 0) F.sgrid = std::max(F.sgrid, 2);          // a chain task and its helpers need two CTAs (see above)
    // epoch-valued flags: counters reach epoch * target and the claim counters epoch * (ntasks + grid); reset before 2^31
    int64_t per_epoch = std::max<int64_t>((int64_t)tasks.size() + F.fgrid, (int64_t)stasks.size() + F.sgrid);
    for (int s = 0; s < ns; ++s) per_epoch = std::max<int64_t>(per_epoch, target[s]);
    const int64_t min_limit = 3 + std::max(0, h->opt.refine_steps);
    h->epoch_limit = (uint32_t)std::max<int64_t>(min_limit, ((int64_t)1 << 31) / per_epoch - 2);
    h->epoch_limit = std::min<uint32_t>(h->epoch_limit, 1u << 19);   // the row-progress words of the factorization hold (call number << 12) | tiles
    if (h->opt.epoch_limit > 0) h->epoch_limit = std::min<uint32_t>(h->epoch_limit, (uint32_t)std::max<int64_t>(min_limit, h->opt.epoch_limit));   // test hook
    return NMPC_OK;
}

// The next call numbers of the factor / solve kernels.  All restart from 1 (all flags zeroed, in stream order) before any
// counter can overflow.  The restart is decided with a margin of all call numbers of one IPM iteration (one factorization, 1 +
// refine_steps solves), so the numbers reserved for one CUDA-graph replay always lie on the same side of a restart.
nmpc_status next_factor_epoch(nmpc_handle_s* h, uint32_t* out) {
    const uint32_t per_iter = 2u + (uint32_t)std::max(0, h->opt.refine_steps);   // one factorization + (1 + refine_steps) solves
    if (std::max(h->epoch_f, std::max(h->epoch_sf, h->epoch_sb)) + per_iter >= h->epoch_limit) {
        CK(cudaMemsetAsync(h->F.sync, 0, (size_t)h->F.sync_words * sizeof(uint32_t), h->stream));
        h->epoch_f = h->epoch_sf = h->epoch_sb = 0;
    }
    *out = ++h->epoch_f;
    return NMPC_OK;
}
// forward / backward call numbers of one solve; a fused solve (backward half only) gets *ef = 0
nmpc_status next_solve_epochs(nmpc_handle_s* h, bool fused, uint32_t* ef, uint32_t* eb) {
    if (std::max(h->epoch_sf, h->epoch_sb) + 1 >= h->epoch_limit) {   // a long run of solves on one factorization: only the solve flags restart
        const size_t off = (size_t)(h->F.sol_done_f - h->F.sync), cnt = (size_t)(h->F.tile_done - h->F.sol_done_f);
        CK(cudaMemsetAsync(h->F.sync + 1, 0, 2 * sizeof(uint32_t), h->stream));
        CK(cudaMemsetAsync(h->F.sync + off, 0, cnt * sizeof(uint32_t), h->stream));
        CK(cudaMemsetAsync(h->F.blk_f, 0, (size_t)(h->F.sub_done - h->F.blk_f) * sizeof(uint32_t), h->stream));
        h->epoch_sf = h->epoch_sb = 0;
    }
    *eb = ++h->epoch_sb;
    *ef = fused ? 0u : ++h->epoch_sf;
    return NMPC_OK;
}

nmpc_status run_factor(nmpc_handle_s* h, double eta, int64_t* info) {
    uint32_t epoch = 0;
    TRY(next_factor_epoch(h, &epoch));
    launch_factor(h->D, h->F, h->d_Kval, eta, epoch, nullptr, h->stream); h->launches += 1;
    int32_t* flag = reinterpret_cast<int32_t*>(h->h_pinned + 16);
    CK(cudaMemcpyAsync(flag, h->D.fail_col, sizeof(int32_t), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    CK(cudaGetLastError());
    h->eta_cur = eta;
    if (*flag != INT_MAX) {
        h->factored = false;
        launch_reset_fail(h->D, h->stream); h->launches += 1;
        if (info) *info = h->S.perm[*flag];
        return NMPC_E_NOT_SPD;
    }
    h->factored = true;
    if (info) *info = -1;
    return NMPC_OK;
}

nmpc_status run_solve(nmpc_handle_s* h, double* rhs, bool fused = false) {       // in place (fused: rhs is written only), async
    uint32_t ef = 0, eb = 0;
    TRY(next_solve_epochs(h, fused, &ef, &eb));
    launch_solve(h->D, h->F, rhs, h->d_x, ef, eb, nullptr, fused, h->stream); h->launches += 1;
    return NMPC_OK;
}
// K^-1 b for the b of the IPM iteration (V.b): with the right-hand-side row b went through the factorization and only the
// backward half runs; else b is copied and solved in place
nmpc_status run_newton_solve(nmpc_handle_s* h) {
    if (h->S.aug) return run_solve(h, h->V.dy, true);
    CK(cudaMemcpyAsync(h->V.dy, h->V.b, sizeof(double) * h->M.n, cudaMemcpyDeviceToDevice, h->stream));
    return run_solve(h, h->V.dy);
}

// One IPM iteration as a CUDA graph (opt.use_graph): parameter upload {mu, tau, call numbers} from pinned memory, S6 (Sigma, rhs),
// a3 (assembly), a4 (factorization), a5 (solves), S8-S10 (step, device-guarded update), then S2 of the NEXT iteration (model
// evaluation, residuals) and the read-back of the reduced scalars + pivot flag.  The kernels take mu / tau / the call numbers
// from device memory (d_par), so the same executable graph is replayed every iteration with one launch.
nmpc_status capture_iteration_graph(nmpc_handle_s* h) {
    const DevModel& M = h->M;
    const IpmVectors& V = h->V;
    cudaStream_t st = h->stream;
    double* hp = h->h_pinned + 24;                       // pinned mirror of d_par
    double* hs = h->h_pinned;
    int32_t* flag = reinterpret_cast<int32_t*>(h->h_pinned + 16);
    const uint32_t* epo = reinterpret_cast<const uint32_t*>(h->d_par + 2);
    cudaGraph_t g = nullptr;
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); h->graph_failed = true; return NMPC_OK; }
    // every captured call is checked; the first failure ends the capture and the plain launch sequence is used instead
    cudaError_t ce = cudaSuccess;
    auto ok = [&](cudaError_t e) { if (ce == cudaSuccess && e != cudaSuccess) ce = e; return ce == cudaSuccess; };
    auto launched = [&]() { return ok(cudaGetLastError()); };
    bool good = ok(cudaMemcpyAsync(h->d_par, hp, 8 * sizeof(double), cudaMemcpyHostToDevice, st));
    if (good) { launch_sigma_rhs(M, V, 0.0, h->d_par, st); good = launched(); }
    if (good) { launch_assemble_K(M, V.Jval, V.Wval, V.sigx, V.q, 0.0, V.Kval, st); good = launched(); }
    if (good) { launch_factor(h->D, h->F, h->d_Kval, 0.0, 0u, epo, st); good = launched(); }
    if (good && !h->S.aug) good = ok(cudaMemcpyAsync(V.dy, V.b, sizeof(double) * M.n, cudaMemcpyDeviceToDevice, st));
    if (good) { launch_solve(h->D, h->F, V.dy, h->d_x, 0u, 0u, epo + 1, h->S.aug, st); good = launched(); }
    if (good) { launch_step(M, V, 0.0, 0.0, h->d_par, st); good = launched(); }
    for (int r = 0; good && r < h->opt.refine_steps; ++r) {      // iterative refinement: solve number r + 1 of this iteration
        launch_refine_residual(M, V, 0.0, h->D.fail_col, st); good = launched();
        if (good) { launch_solve(h->D, h->F, V.rho, h->d_x, 0u, 0u, epo + 3 + 2 * r, false, st); good = launched(); }
        if (good) { launch_add_correction(M, V, h->D.fail_col, st); good = launched(); }
        if (good) { launch_step(M, V, 0.0, 0.0, h->d_par, st); good = launched(); }
    }
    if (good) { launch_update(M, V, h->D.fail_col, st); good = launched(); }
    if (good) { launch_model_eval(M, V.y, V.wp, V.wm, nullptr, V.c, V.gradf, V.Jval, V.Wval, st); good = launched(); }
    if (good) { launch_residuals(M, V, h->opt.gamma, st); good = launched(); }
    if (good) good = ok(cudaMemcpyAsync(hs, V.scal, sizeof(double) * 10, cudaMemcpyDeviceToHost, st));
    if (good) good = ok(cudaMemcpyAsync(flag, h->D.fail_col, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    const cudaError_t ee = cudaStreamEndCapture(st, &g);
    if (!good || ee != cudaSuccess || !g) {
        cudaGetLastError();
        if (g) cudaGraphDestroy(g);
        h->err = std::string("CUDA-graph capture of the IPM iteration failed (") + cudaGetErrorString(good ? ee : ce) + "); using plain launches";
        h->graph_failed = true;
        return NMPC_OK;
    }
    if (cudaGraphInstantiate(&h->iter_graph, g, 0) != cudaSuccess) { cudaGetLastError(); h->iter_graph = nullptr; h->graph_failed = true; }
    cudaGraphDestroy(g);
    return NMPC_OK;
}

struct PhaseTimer {                 // optional CUDA-event phase timing (opt.time_phases): sums per solve and per iteration
    nmpc_handle_s* h; bool on; double* acc = nullptr; double* acc_it = nullptr;
    double it_ms[5] = {0, 0, 0, 0, 0};   // eval, assemble, factor, solve, vector of the iteration being built
    void begin(double* a, int phase) { if (!on) return; acc = a; acc_it = it_ms + phase; cudaEventRecord(h->ev[0], h->stream); }
    void end() {
        if (!on || !acc) return;
        cudaEventRecord(h->ev[1], h->stream); cudaEventSynchronize(h->ev[1]);
        float ms = 0; cudaEventElapsedTime(&ms, h->ev[0], h->ev[1]); *acc += ms; *acc_it += ms; acc = nullptr;
    }
    void flush(nmpc_trace_row* row) {    // S2 of iteration k+1 is booked on iteration k (as in the graph replay)
        if (row) { row->ms_eval = it_ms[0]; row->ms_assemble = it_ms[1]; row->ms_factor = it_ms[2]; row->ms_solve = it_ms[3]; row->ms_vector = it_ms[4]; }
        for (double& v : it_ms) v = 0.0;
    }
};

}  // namespace

extern "C" {

nmpc_status nmpc_analyze(const nmpc_pattern* pattern, const nmpc_ocp* ocp, const nmpc_options* opt, void* cuda_stream, nmpc_handle* out) {
    if (!out) return NMPC_E_ARG;
    *out = nullptr;
    g_create_error.clear();
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); g_create_error = "no CUDA device"; return NMPC_E_CUDA; }
    nmpc_handle_s* h = new (std::nothrow) nmpc_handle_s();
    if (!h) return NMPC_E_ALLOC;
    auto fail = [&](nmpc_status s) { g_create_error = h->err; nmpc_destroy(h); return s; };
    if (opt) h->opt = *opt; else default_options(&h->opt);
    if (h->opt.mu_warm <= 0.0) h->opt.mu_warm = h->opt.eps_outer / 10.0;
    h->opt.refine_steps = std::min(4, std::max(0, h->opt.refine_steps));
    int smem_optin = 0, num_sms = 0, lat_ctas = 1, lat_rmax = 0;
    size_t lat_smem = 0;
    if (cudaGetDevice(&h->dev) != cudaSuccess || cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, h->dev) != cudaSuccess ||
        configure_factor_kernels(smem_optin, true, &lat_ctas, &lat_smem, &lat_rmax) != cudaSuccess) {
        h->err = std::string("device query failed: ") + cudaGetErrorString(cudaGetLastError()); return fail(NMPC_E_CUDA);
    }
    h->stream = (cudaStream_t)cuda_stream;
    if (!h->stream) {
        // the legacy default stream cannot be captured into a graph: use an own BLOCKING stream, which keeps the implicit
        // ordering with work the caller issues on the legacy default stream (e.g. torch's default stream)
        if (cudaStreamCreate(&h->stream) != cudaSuccess) { h->err = "cudaStreamCreate failed"; cudaGetLastError(); return fail(NMPC_E_CUDA); }
        h->own_stream = true;
    }
    // The amalgamation threshold on auto (relax_small < 0): dependency hops, not flops, bound most of the path (DESIGN.md section
    // 6.2), so supernodes are merged more aggressively than the classical default of 8: 64 in general (C4: 6565 -> 1230 fronts,
    // nnz(L) +30 % but factor + solve -9 %), 32 with dissection leaves of 32 for a small problem that is then eligible for the
    // latency mode below (C1: 8 -> 7 levels, 436 -> 189 fronts).  Latency mode = every front fits ONE CTA's shared memory
    // (lat_rmax rows, computed from the device's shared-memory size) and sum cc^2 <= 1e8.  The small-problem analysis is tried
    // first when n is small, so C0/C1-class problems are analysed once; only a problem that turns out not to be eligible (or a
    // large-n problem that turns out to be) pays for a second analysis.
    const bool auto_relax = h->opt.relax_small < 0 && h->opt.smem_front_max <= 0;
    auto eligible = [&](const Symbolic& S) { return S.flops <= 1e8 && S.max_front <= lat_rmax; };
    auto analyze_with = [&](bool small_variant, Symbolic& S) -> nmpc_status {
        nmpc_options o = h->opt;
        if (o.relax_small < 0) o.relax_small = small_variant ? 32 : 64;
        if (small_variant && o.nd_leaf <= 0) o.nd_leaf = 32;      // smaller dissection leaves: C1 factor + solve another -11 %
        const bool augment = o.fuse_rhs > 0 || (o.fuse_rhs < 0 && ocp && ocp->model != NMPC_MODEL_NONE);
        try { return analyze_symbolic(pattern, ocp, &o, S, augment); }
        catch (const std::bad_alloc&) { S.error = "host allocation failed"; return NMPC_E_ALLOC; }
    };
    const int64_t n_hint = pattern ? pattern->n : (ocp ? (int64_t)ocp->N * (ocp->nx + ocp->nu) : 0);
    const bool small_first = auto_relax && n_hint <= 8192;
    nmpc_status st = analyze_with(small_first, h->S);
    if (st != NMPC_OK) { h->err = h->S.error; return fail(st); }
    if (auto_relax && small_first != eligible(h->S)) {
        Symbolic S2;
        if (analyze_with(!small_first, S2) == NMPC_OK && (small_first || eligible(S2))) { S2.analyze_ms += h->S.analyze_ms; h->S = std::move(S2); }
    }
    auto body = [&]() -> nmpc_status {
        const Symbolic& S = h->S;
        int ctas_per_sm = lat_ctas, small_max_r = lat_rmax;
        size_t factor_smem = lat_smem;
        // latency mode: a small problem (dependency-latency bound) whose largest fronts fit the whole
        // shared memory of an SM keeps every front in the one-CTA kernel family; else two CTAs per SM and tiled big fronts
        const bool latency_mode = eligible(S) && h->opt.smem_front_max <= 0;
        if (!latency_mode) CK(configure_factor_kernels(smem_optin, false, &ctas_per_sm, &factor_smem, &small_max_r));
        if (h->opt.smem_front_max > 0) small_max_r = std::min(small_max_r, h->opt.smem_front_max);
        int solve_ctas = 1, sbuf = 0; size_t solve_smem = 0;
        CK(configure_solve_kernels(smem_optin, small_max_r, &solve_ctas, &solve_smem, &sbuf));
        h->F.sbuf = sbuf;
        DevSym& D = h->D;
        D.ns = S.ns; D.n = S.n; D.aug_col = S.aug ? (int32_t)S.n : -1;
        TRY(upload(h, S.sn_start, &D.sn_start)); TRY(upload(h, S.rows_ptr, &D.rows_ptr)); TRY(upload(h, S.rows, &D.rows));
        TRY(upload(h, S.child_ptr, &D.child_ptr)); TRY(upload(h, S.child_idx, &D.child_idx));
        TRY(upload(h, S.rel_ptr, &D.rel_ptr)); TRY(upload(h, S.rel, &D.rel));
        TRY(upload(h, S.panel_ptr, &D.panel_ptr)); TRY(upload(h, S.upd_ptr, &D.upd_ptr));
        TRY(upload(h, S.kent_ptr, &D.kent_ptr));                 // kent_src / kent_dst: per front class, in build_plan
        TRY(upload(h, S.perm, &D.perm));
        TRY(dalloc(h, (size_t)S.panel_ptr.back() + 4 * TILE, &D.L)); TRY(dalloc(h, (size_t)S.upd_ptr.back(), &D.U, false));
        TRY(dalloc(h, (size_t)S.rel_ptr.back(), &D.ctr)); TRY(dalloc(h, 1, &D.fail_col));
        TRY(dalloc(h, (size_t)S.nt, &D.dinv));
        launch_reset_fail(D, h->stream);
        TRY(dalloc(h, (size_t)S.nnzKa, &h->d_Kval)); TRY(dalloc(h, (size_t)S.nt, &h->d_x));   // [K values | b | 0] with the right-hand-side row
        TRY(build_plan(h, small_max_r, ctas_per_sm, factor_smem, solve_ctas, solve_smem, num_sms));
        // symmetric CSR of K for nmpc_kkt_multiply
        {
            const int64_t n = S.n;
            std::vector<int64_t> ptr(n + 1, 0);
            for (int64_t i = 0; i < n; ++i)
                for (int64_t p = S.K.ptr[i]; p < S.K.ptr[i + 1]; ++p) { ptr[i + 1]++; if (S.K.idx[p] != i) ptr[S.K.idx[p] + 1]++; }
            for (int64_t i = 0; i < n; ++i) ptr[i + 1] += ptr[i];
            std::vector<int32_t> idx(ptr[n]), src(ptr[n]);
            std::vector<int64_t> pos(ptr.begin(), ptr.end() - 1);
            for (int64_t i = 0; i < n; ++i)
                for (int64_t p = S.K.ptr[i]; p < S.K.ptr[i + 1]; ++p) {
                    const int32_t j = S.K.idx[p];
                    idx[pos[i]] = j; src[pos[i]++] = (int32_t)p;
                    if (j != i) { idx[pos[j]] = (int32_t)i; src[pos[j]++] = (int32_t)p; }
                }
            const int64_t* tp = nullptr; const int32_t* ti = nullptr;
            TRY(upload(h, ptr, &tp)); h->d_full_ptr = const_cast<int64_t*>(tp);
            TRY(upload(h, idx, &ti)); h->d_full_idx = const_cast<int32_t*>(ti);
            TRY(upload(h, src, &ti)); h->d_full_src = const_cast<int32_t*>(ti);
        }
        size_t pinned = 64;
        if (S.mm.present) {
            const ModelMaps& mm = S.mm;
            DevModel& M = h->M;
            h->has_model = true;
            M.desc = mm.desc; M.n = mm.n; M.m = mm.m; M.nnzJ = mm.J.nnz(); M.nnzW = mm.W.nnz(); M.nnzK = mm.K.nnz();
            TRY(upload(h, mm.J.ptr, &M.J_ptr)); TRY(upload(h, mm.J.idx, &M.J_idx));
            TRY(upload(h, mm.jt_ptr, &M.jt_ptr)); TRY(upload(h, mm.jt_idx, &M.jt_idx)); TRY(upload(h, mm.jt_row, &M.jt_row));
            TRY(upload(h, mm.trip_ptr, &M.trip_ptr)); TRY(upload(h, mm.trip_a, &M.trip_a)); TRY(upload(h, mm.trip_b, &M.trip_b)); TRY(upload(h, mm.trip_r, &M.trip_r));
            TRY(upload(h, mm.k_w, &M.k_w)); TRY(upload(h, mm.k_diag, &M.k_diag));
            const int nv = mm.desc.nv;
            std::vector<double> lb(mm.n), ub(mm.n), ui(std::max(1, mm.desc.nu), 0.0);
            // row intervals: the gamma tube of Eq. (16) around every equality row (dynamics, general rows with lo == hi), the
            // stated interval for the inequality rows; an infinite side has no slack and no multiplier
            std::vector<double> cl(mm.m), cu(mm.m);
            h->nmult = 0;
            for (int64_t r = 0; r < mm.m; ++r) {
                const bool eq = mm.cl[r] == mm.cu[r];
                cl[r] = eq ? mm.cl[r] - h->opt.gamma : mm.cl[r]; cu[r] = eq ? mm.cu[r] + h->opt.gamma : mm.cu[r];
                h->nmult += (int)std::isfinite(cl[r]) + (int)std::isfinite(cu[r]);
                if (!std::isfinite(cl[r]) && !std::isfinite(cu[r])) { h->err = "general row without a finite bound"; return NMPC_E_ARG; }
            }
            M.m_dyn = mm.m_dyn;
            TRY(upload(h, cl, &M.cl)); TRY(upload(h, cu, &M.cu)); TRY(upload(h, mm.g_val, &M.g_val));
            for (int64_t i = 0; i < mm.n; ++i) {
                lb[i] = ocp->lb ? ocp->lb[i % nv] : -INFINITY; ub[i] = ocp->ub ? ocp->ub[i % nv] : INFINITY;
                if (std::isfinite(lb[i])) h->nmult++;
                if (std::isfinite(ub[i])) h->nmult++;
                if (!(lb[i] < ub[i])) { h->err = "lb >= ub"; return NMPC_E_ARG; }
            }
            for (int a = 0; a < mm.desc.nu; ++a) ui[a] = ocp->u_init ? ocp->u_init[a] : 0.0;
            TRY(upload(h, lb, &M.lb)); TRY(upload(h, ub, &M.ub));
            const double* tu = nullptr; TRY(upload(h, ui, &tu)); h->d_uinit = const_cast<double*>(tu);
            TRY(dalloc(h, (size_t)mm.desc.nx, &M.x0)); TRY(dalloc(h, (size_t)std::max<int64_t>(1, (int64_t)mm.desc.N * mm.desc.nr), &M.ref));
            IpmVectors& V = h->V;
            const size_t n = mm.n, m = mm.m;
            TRY(dalloc(h, n, &V.y)); TRY(dalloc(h, m, &V.sp)); TRY(dalloc(h, m, &V.sm)); TRY(dalloc(h, m, &V.wp)); TRY(dalloc(h, m, &V.wm));
            TRY(dalloc(h, n, &V.zL)); TRY(dalloc(h, n, &V.zU)); TRY(dalloc(h, m, &V.c)); TRY(dalloc(h, n, &V.gradf));
            TRY(dalloc(h, (size_t)M.nnzJ, &V.Jval)); TRY(dalloc(h, (size_t)M.nnzW, &V.Wval));
            V.Kval = h->d_Kval;
            TRY(dalloc(h, m, &V.r_pp)); TRY(dalloc(h, m, &V.r_pm)); TRY(dalloc(h, m, &V.q)); TRY(dalloc(h, m, &V.t));
            TRY(dalloc(h, n, &V.sigx)); TRY(dalloc(h, n, &V.dy));
            if (S.aug) V.b = h->d_Kval + S.nnzK;              // the right-hand side of Eq. (17) is written straight into the factorization's value array
            else TRY(dalloc(h, n, &V.b));
            TRY(dalloc(h, m, &V.dsp)); TRY(dalloc(h, m, &V.dsm)); TRY(dalloc(h, m, &V.dwp)); TRY(dalloc(h, m, &V.dwm));
            TRY(dalloc(h, n, &V.dzL)); TRY(dalloc(h, n, &V.dzU));
            TRY(dalloc(h, (size_t)RED_BLOCKS * 8, &V.partial)); TRY(dalloc(h, (size_t)NSCAL, &V.scal));
            TRY(dalloc(h, 8, &h->d_par));
            TRY(dalloc(h, n, &V.rho)); TRY(dalloc(h, n, &V.yt)); TRY(dalloc(h, m, &V.ct));
            {   // symmetric CSR of W (lower CSR in value order) for the W dy product of the refinement residual
                std::vector<int64_t> ptr(n + 1, 0);
                for (int64_t i = 0; i < (int64_t)n; ++i)
                    for (int64_t p = mm.W.ptr[i]; p < mm.W.ptr[i + 1]; ++p) { ptr[i + 1]++; if (mm.W.idx[p] != i) ptr[mm.W.idx[p] + 1]++; }
                for (size_t i = 0; i < n; ++i) ptr[i + 1] += ptr[i];
                std::vector<int32_t> idx(ptr[n]), src(ptr[n]);
                std::vector<int64_t> pos(ptr.begin(), ptr.end() - 1);
                for (int64_t i = 0; i < (int64_t)n; ++i)
                    for (int64_t p = mm.W.ptr[i]; p < mm.W.ptr[i + 1]; ++p) {
                        const int32_t j = mm.W.idx[p];
                        idx[pos[i]] = j; src[pos[i]++] = (int32_t)p;
                        if (j != i) { idx[pos[j]] = (int32_t)i; src[pos[j]++] = (int32_t)p; }
                    }
                TRY(upload(h, ptr, &M.wf_ptr)); TRY(upload(h, idx, &M.wf_idx)); TRY(upload(h, src, &M.wf_src));
            }
            pinned += (size_t)mm.desc.nx + (size_t)mm.desc.N * mm.desc.nr + n;
        }
        h->pinned_doubles = pinned;
        CK(cudaMallocHost((void**)&h->h_pinned, pinned * sizeof(double)));
        CK(cudaEventCreate(&h->ev[0])); CK(cudaEventCreate(&h->ev[1]));
        CK(cudaStreamSynchronize(h->stream));
        return NMPC_OK;
    };
    st = body();
    if (st != NMPC_OK) return fail(st);
    *out = h;
    return NMPC_OK;
}

void nmpc_destroy(nmpc_handle h) {
    if (!h) return;
    DeviceGuard dg(h);
    for (void* p : h->allocs) cudaFree(p);
    if (h->h_pinned) cudaFreeHost(h->h_pinned);
    if (h->iter_graph) cudaGraphExecDestroy(h->iter_graph);
    if (h->ev[0]) cudaEventDestroy(h->ev[0]);
    if (h->ev[1]) cudaEventDestroy(h->ev[1]);
    for (cudaEvent_t e : h->it_ev) cudaEventDestroy(e);
    if (h->own_stream) cudaStreamDestroy(h->stream);
    delete h;
}

#ifdef NMPC_TRACE_BUILD
int64_t nmpc_get_task_trace(nmpc_handle h, int32_t kind, int32_t* tasks_host, uint64_t* stamps_host, int64_t cap) {
    if (!h || kind < 0 || kind > 2) return -1;
    DeviceGuard dg(h);
    if (kind == 2) {                                     // phase cycles of the diagonal-tile POTRFs since the last read (8 words)
        if (!stamps_host || cap < 8) return 8;
        if (cudaStreamSynchronize(h->stream) != cudaSuccess || read_potrf_cycles(reinterpret_cast<unsigned long long*>(stamps_host), true) != cudaSuccess) return -1;
        return 8;
    }
    const int64_t nt = kind == 0 ? h->F.n_ftasks : h->F.n_stasks;
    const unsigned long long* tr = kind == 0 ? h->F.ftrace : h->F.strace;
    if (!tr) return 0;
    if (!tasks_host || !stamps_host) return nt;
    const int64_t k = std::min(nt, cap);
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) return -1;
    if (cudaMemcpy(tasks_host, kind == 0 ? h->F.ftasks : h->F.stasks, (size_t)k * sizeof(int4), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    if (cudaMemcpy(stamps_host, tr, (size_t)k * 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return k;
}
#endif

const char* nmpc_last_error(nmpc_handle h) { return h ? h->err.c_str() : g_create_error.c_str(); }
int64_t nmpc_launch_count(nmpc_handle h) { return h ? h->launches : 0; }

nmpc_status nmpc_get_info(nmpc_handle h, nmpc_sym_info* out) {
    if (!h || !out) return NMPC_E_ARG;
    nmpc_fill_info(h->S, out);
    out->n_large_fronts = h->n_big_fronts;
    return NMPC_OK;
}

nmpc_status nmpc_get_factor(nmpc_handle h, double* panels_host) {
    if (!h || !panels_host) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->factored) { h->err = "no successful factorization"; return NMPC_E_STATE; }
    const Symbolic& S = h->S;
    if (!S.aug) {
        CK(cudaMemcpyAsync(panels_host, h->D.L, (size_t)S.panel_ptr.back() * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CK(cudaStreamSynchronize(h->stream));
        return NMPC_OK;
    }
    // with the right-hand-side row: repack without that row / pivot (the layout nmpc_get_info describes)
    std::vector<double> all;
    try { all.resize((size_t)S.panel_ptr.back()); } catch (const std::bad_alloc&) { h->err = "host allocation failed"; return NMPC_E_ALLOC; }
    CK(cudaMemcpy(all.data(), h->D.L, all.size() * sizeof(double), cudaMemcpyDeviceToHost));
    int64_t off = 0;
    for (int32_t s = 0; s < S.ns; ++s) {
        const int64_t r = S.rows_ptr[s + 1] - S.rows_ptr[s], ld = panel_ld(r);
        const int64_t rv = S.v_rows_ptr[s + 1] - S.v_rows_ptr[s], wv = S.v_sn_start[s + 1] - S.v_sn_start[s], ldv = panel_ld(rv);
        // the row left out is the last one of the front; in the supernode that holds its pivot it is the last column as well
        for (int64_t j = 0; j < wv; ++j) {
            const double* src = all.data() + S.panel_ptr[s] + j * ld;
            double* dst = panels_host + off + j * ldv;
            for (int64_t i = 0; i < rv; ++i) dst[i] = src[i];
            if (ldv > rv) dst[rv] = 0.0;
        }
        off += ldv * wv;
    }
    return NMPC_OK;
}

nmpc_status nmpc_factor(nmpc_handle h, const double* values_dev, double eta, int64_t* info_host) {
    if (!h || !values_dev) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (values_dev != h->d_Kval)
        CK(cudaMemcpyAsync(h->d_Kval, values_dev, (size_t)h->S.nnzK * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    h->rhs_row_valid = false;
    return run_factor(h, eta, info_host);
}

nmpc_status nmpc_factor_rhs(nmpc_handle h, const double* values_dev, const double* rhs_dev, double eta, int64_t* info_host) {
    if (!h || !values_dev || !rhs_dev) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->S.aug) { h->err = "nmpc_factor_rhs needs a handle created with options.fuse_rhs"; return NMPC_E_STATE; }
    if (values_dev != h->d_Kval)
        CK(cudaMemcpyAsync(h->d_Kval, values_dev, (size_t)h->S.nnzK * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    if (rhs_dev != h->d_Kval + h->S.nnzK)
        CK(cudaMemcpyAsync(h->d_Kval + h->S.nnzK, rhs_dev, (size_t)h->S.n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    const nmpc_status st = run_factor(h, eta, info_host);
    h->rhs_row_valid = st == NMPC_OK;
    return st;
}

nmpc_status nmpc_solve_fused(nmpc_handle h, double* out_dev) {
    if (!h || !out_dev) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->S.aug || !h->factored || !h->rhs_row_valid) { h->err = "nmpc_solve_fused needs a successful nmpc_factor_rhs"; return NMPC_E_STATE; }
    TRY(run_solve(h, out_dev, true));
    CK(cudaGetLastError());
    return NMPC_OK;
}

nmpc_status nmpc_solve(nmpc_handle h, double* rhs, int32_t nrhs) {
    if (!h || !rhs || nrhs < 1) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->factored) { h->err = "nmpc_solve before a successful nmpc_factor"; return NMPC_E_STATE; }
    for (int k = 0; k < nrhs; ++k) TRY(run_solve(h, rhs + (int64_t)k * h->S.n));
    CK(cudaGetLastError());
    return NMPC_OK;
}

// ---- nmpc_solve_static: the two-sided solve with its work vector in a file-scope device array (no allocation anywhere on the
//      path, not even at analysis time, for this vector).  The array is part of the library image: every GPU that loads the
//      library holds NMPC_STATIC_SOLVE_DOUBLES * 8 bytes = 2 MiB of it until the process exits.  In host code the NAME of the
//      array is a host-side stand-in, not a device address; the device address comes from cudaGetSymbolAddress, once per
//      device with that device current (static_solve_scratch), and THAT pointer goes to the kernel.  Every call on a device
//      shares the array, which keeps the last call's contents: the part a call uses is cleared first, and calls that overlap
//      on the GPU (two streams, two handles) race. ----
#define NMPC_STATIC_SOLVE_DOUBLES_IMPL 262144
static_assert(NMPC_STATIC_SOLVE_DOUBLES_IMPL == NMPC_STATIC_SOLVE_DOUBLES, "include/nmpc.h states the size of the static work vector");
static __device__ __align__(256) double g_static_solve_x[NMPC_STATIC_SOLVE_DOUBLES_IMPL];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
double* g_static_ptr[STATIC_MAX_DEVICES] = {};            // device address of g_static_solve_x per device ordinal (0: not looked up yet)

// the handle's device is current (DeviceGuard of the caller)
nmpc_status static_solve_scratch(nmpc_handle_s* h, double** out) {
    if (h->dev < 0 || h->dev >= STATIC_MAX_DEVICES) { h->err = "nmpc_solve_static: device ordinal beyond " + std::to_string(STATIC_MAX_DEVICES - 1); return NMPC_E_ARG; }
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[h->dev]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_solve_x);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            h->err = std::string("nmpc_solve_static: cudaGetSymbolAddress failed (") + cudaGetErrorString(e) + ")";
            return NMPC_E_CUDA;
        }
        g_static_ptr[h->dev] = p;
    }
    *out = g_static_ptr[h->dev];
    return NMPC_OK;
}
}  // namespace

nmpc_status nmpc_solve_static(nmpc_handle h, const double* rhs_dev, double* out_dev) {
    if (!h || !rhs_dev || !out_dev) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if ((int64_t)h->S.nt > (int64_t)NMPC_STATIC_SOLVE_DOUBLES) {
        h->err = "nmpc_solve_static: the structure needs a work vector of " + std::to_string((long long)h->S.nt) + " doubles, the static one holds " +
                 std::to_string((long long)NMPC_STATIC_SOLVE_DOUBLES) + " (NMPC_STATIC_SOLVE_DOUBLES); use nmpc_solve";
        return NMPC_E_ARG;
    }
    if (!h->factored) { h->err = "nmpc_solve_static before a successful nmpc_factor"; return NMPC_E_STATE; }
    double* xs = nullptr;
    TRY(static_solve_scratch(h, &xs));
    // the array keeps what the last call left (possibly of another handle): the part this call uses starts at zero, like the
    // handle's own work vector did after nmpc_analyze
    CK(cudaMemsetAsync(xs, 0, sizeof(double) * (size_t)h->S.nt, h->stream));
    if (out_dev != rhs_dev) CK(cudaMemcpyAsync(out_dev, rhs_dev, sizeof(double) * (size_t)h->S.n, cudaMemcpyDeviceToDevice, h->stream));
    uint32_t ef = 0, eb = 0;
    TRY(next_solve_epochs(h, false, &ef, &eb));
    launch_solve(h->D, h->F, out_dev, xs, ef, eb, nullptr, false, h->stream); h->launches += 1;
    CK(cudaGetLastError());
    return NMPC_OK;
}

nmpc_status nmpc_kkt_multiply(nmpc_handle h, const double* x_dev, double* y_dev) {
    if (!h || !x_dev || !y_dev) return NMPC_E_ARG;
    DeviceGuard dg(h);
    launch_kkt_multiply(h->S.n, h->d_full_ptr, h->d_full_idx, h->d_full_src, h->d_Kval, h->eta_cur, x_dev, y_dev, h->stream);
    h->launches++;
    CK(cudaGetLastError());
    return NMPC_OK;
}

nmpc_status nmpc_update_params(nmpc_handle h, const double* x0_dev, const double* ref_dev) {
    if (!h) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) { h->err = "handle has no model"; return NMPC_E_STATE; }
    const ModelDesc& d = h->M.desc;
    if (x0_dev) CK(cudaMemcpyAsync(h->M.x0, x0_dev, sizeof(double) * d.nx, cudaMemcpyDeviceToDevice, h->stream));
    if (ref_dev && d.nr > 0) CK(cudaMemcpyAsync(h->M.ref, ref_dev, sizeof(double) * (size_t)d.N * d.nr, cudaMemcpyDeviceToDevice, h->stream));
    return NMPC_OK;
}

nmpc_status nmpc_update_params_host(nmpc_handle h, const double* x0_host, const double* ref_host) {
    if (!h) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) { h->err = "handle has no model"; return NMPC_E_STATE; }
    const ModelDesc& d = h->M.desc;
    double* stage = h->h_pinned + 64;
    CK(cudaStreamSynchronize(h->stream));               // staging buffer reuse
    if (x0_host) {
        std::memcpy(stage, x0_host, sizeof(double) * d.nx);
        CK(cudaMemcpyAsync(h->M.x0, stage, sizeof(double) * d.nx, cudaMemcpyHostToDevice, h->stream));
    }
    if (ref_host && d.nr > 0) {
        double* s2 = stage + d.nx;
        std::memcpy(s2, ref_host, sizeof(double) * (size_t)d.N * d.nr);
        CK(cudaMemcpyAsync(h->M.ref, s2, sizeof(double) * (size_t)d.N * d.nr, cudaMemcpyHostToDevice, h->stream));
    }
    return NMPC_OK;
}

nmpc_status nmpc_get_iterate(nmpc_handle h, double* y, double* sp, double* sm, double* wp, double* wm, double* zL, double* zU) {
    if (!h) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) return NMPC_E_STATE;
    const size_t n = h->M.n * sizeof(double), m = h->M.m * sizeof(double);
    const IpmVectors& V = h->V;
    if (y) CK(cudaMemcpyAsync(y, V.y, n, cudaMemcpyDeviceToDevice, h->stream));
    if (sp) CK(cudaMemcpyAsync(sp, V.sp, m, cudaMemcpyDeviceToDevice, h->stream));
    if (sm) CK(cudaMemcpyAsync(sm, V.sm, m, cudaMemcpyDeviceToDevice, h->stream));
    if (wp) CK(cudaMemcpyAsync(wp, V.wp, m, cudaMemcpyDeviceToDevice, h->stream));
    if (wm) CK(cudaMemcpyAsync(wm, V.wm, m, cudaMemcpyDeviceToDevice, h->stream));
    if (zL) CK(cudaMemcpyAsync(zL, V.zL, n, cudaMemcpyDeviceToDevice, h->stream));
    if (zU) CK(cudaMemcpyAsync(zU, V.zU, n, cudaMemcpyDeviceToDevice, h->stream));
    return NMPC_OK;
}

nmpc_status nmpc_set_iterate(nmpc_handle h, const double* y, const double* sp, const double* sm, const double* wp, const double* wm, const double* zL, const double* zU) {
    if (!h || !y || !sp || !sm || !wp || !wm || !zL || !zU) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) return NMPC_E_STATE;
    const size_t n = h->M.n * sizeof(double), m = h->M.m * sizeof(double);
    const IpmVectors& V = h->V;
    CK(cudaMemcpyAsync(V.y, y, n, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(V.sp, sp, m, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(V.sm, sm, m, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(V.wp, wp, m, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(V.wm, wm, m, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(V.zL, zL, n, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(V.zU, zU, n, cudaMemcpyDeviceToDevice, h->stream));
    h->have_state = true;
    return NMPC_OK;
}

nmpc_status nmpc_model_eval(nmpc_handle h, const double* y, const double* lam, double* c, double* gradf, double* Jval, double* Wval) {
    if (!h || !y) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) return NMPC_E_STATE;
    if (Wval && !lam) return NMPC_E_ARG;
    launch_model_eval(h->M, y, nullptr, nullptr, lam, c, gradf, Jval, Wval, h->stream);
    h->launches++;
    CK(cudaGetLastError());
    return NMPC_OK;
}

nmpc_status nmpc_assemble(nmpc_handle h, const double* Jval, const double* Wval, const double* sigx, const double* q, double eta, double* Kval) {
    if (!h || !Jval || !Wval || !sigx || !q || !Kval) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) return NMPC_E_STATE;
    launch_assemble_K(h->M, Jval, Wval, sigx, q, eta, Kval, h->stream);
    h->launches++;
    CK(cudaGetLastError());
    return NMPC_OK;
}

nmpc_status nmpc_get_jac_pattern(nmpc_handle h, int64_t* nnz, int64_t* rowptr, int32_t* colind) {
    if (!h) return NMPC_E_ARG;
    if (!h->has_model) return NMPC_E_STATE;
    return nmpc_copy_pattern_internal(h->S.mm.J, nnz, rowptr, colind);
}
nmpc_status nmpc_get_hess_pattern(nmpc_handle h, int64_t* nnz, int64_t* rowptr, int32_t* colind) {
    if (!h) return NMPC_E_ARG;
    if (!h->has_model) return NMPC_E_STATE;
    return nmpc_copy_pattern_internal(h->S.mm.W, nnz, rowptr, colind);
}
nmpc_status nmpc_get_kkt_pattern(nmpc_handle h, int64_t* nnz, int64_t* rowptr, int32_t* colind) {
    if (!h) return NMPC_E_ARG;
    return nmpc_copy_pattern_internal(h->S.K, nnz, rowptr, colind);
}

// ---- Algorithm 2 (LiftedIPM), steps S1..S10 of DESIGN.md section 3 ----
nmpc_status nmpc_ipm_solve(nmpc_handle h, int32_t warm, int32_t use_y0, double* y_inout, nmpc_stats* stats, nmpc_trace_row* trace, int32_t trace_cap) {
    if (!h) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) { h->err = "nmpc_ipm_solve needs a model (nmpc_ocp)"; return NMPC_E_STATE; }
    if (use_y0 && !y_inout) return NMPC_E_ARG;
    const nmpc_options& o = h->opt;
    const DevModel& M = h->M;
    const IpmVectors& V = h->V;
    cudaStream_t st = h->stream;
    auto t_begin = std::chrono::steady_clock::now();
    nmpc_stats S{};
    PhaseTimer pt{h, o.time_phases != 0 && stats != nullptr};
    double mu;
    if (warm && h->have_state) {                                               // S1 warm: z <- z* (Alg. 1 line 10)
        launch_warm_push(M, V, o.warm_push, st); h->launches++;
        mu = o.mu_warm;
    } else {                                                                   // S1 cold
        if (use_y0) CK(cudaMemcpyAsync(V.y, y_inout, sizeof(double) * M.n, cudaMemcpyDeviceToDevice, st));
        launch_cold_init_y(M, V, h->d_uinit, use_y0, o.kappa_push, o.mu0, st);
        launch_model_eval(M, V.y, nullptr, nullptr, nullptr, V.c, nullptr, nullptr, nullptr, st);
        launch_cold_init_s(M, V, o.gamma, o.s_floor, o.mu0, st);
        h->launches += 3;
        mu = o.mu0;
    }
    double eta_last = 0.0, E0 = 0.0;
    int it = 0, nfact = 0, retries = 0;
    nmpc_status status = NMPC_E_MAXITER;
    double* hs = h->h_pinned;
    // Without phase timing the factorization's pivot flag is NOT read back right after the factorization: the solve, the
    // step and the (device-guarded) update are enqueued behind it and the flag travels with the next iteration's residual
    // scalars -- one host synchronisation per IPM iteration.  A failed pivot leaves the iterate untouched (update_kernel
    // checks the flag), so the inertia-correction retry below starts from exactly the state of the synchronous flow.
    const bool async = !o.time_phases && !o.globalization;   // the line search reads merit values back: synchronous flow
    if (async && o.use_graph && !h->iter_graph && !h->graph_failed) TRY(capture_iteration_graph(h));
    const bool graph = async && o.use_graph && h->iter_graph != nullptr;
    // traced solves: one CUDA event per iteration, recorded (no synchronisation) right before the iteration's S6 is launched
    const int n_ev = trace ? std::min(trace_cap, o.max_iter) + 1 : 0;
    while ((int)h->it_ev.size() < n_ev) { cudaEvent_t e = nullptr; CK(cudaEventCreate(&e)); h->it_ev.push_back(e); }
    auto mark_iteration = [&](int k) {                   // start of iteration k = end of iteration k-1
        if (k < n_ev) cudaEventRecord(h->it_ev[k], st);
        pt.flush(trace && k > 0 && k - 1 < trace_cap ? &trace[k - 1] : nullptr);
    };
    bool top_done = false;                               // the previous graph replay already ran S2 + the read-back
    bool pending = false;                                // a factorization whose flag has not been checked yet
    double pend_mu = 0.0, pend_tau = 0.0;
    int32_t* flag = reinterpret_cast<int32_t*>(h->h_pinned + 16);
    auto retry_with_eta = [&](double& eta) -> nmpc_status {   // S7: inertia correction, Eq. (13)/(15); synchronous
        while (true) {
            ++retries;
            if (eta == 0.0) eta = (eta_last == 0.0) ? o.eta_first : std::max(o.eta_min, o.eta_shrink * eta_last);
            else eta = ((eta_last == 0.0) ? o.eta_grow_first : o.eta_grow) * eta;
            if (eta > o.eta_max) return NMPC_E_INERTIA;
            ++nfact;
            pt.begin(&S.ms_factor, 2);
            nmpc_status fs = run_factor(h, eta, nullptr);
            pt.end();
            if (fs == NMPC_OK) return NMPC_OK;
            if (fs != NMPC_E_NOT_SPD) return fs;
        }
    };
    // ---- filter line search on the primal step (options.globalization; ref. [17] Algorithm A, steps A-5.1 .. A-5.10 and A-7,
    //      reading G20 of DESIGN.md section 3): theta and phi_mu of the trial points are reduced on the device, the filter
    //      (a short list of pairs) and the acceptance tests are host scalars ----
    std::vector<std::pair<double, double>> flt;
    double th_max = 0.0, th_min = 0.0, flt_mu = -1.0;
    bool flt_ready = false;
    int last_backtracks = 0;
    double* hm = h->h_pinned + 40;                        // pinned: merit scalars [0..4], step lengths [5..6], accepted alpha [7]
    struct Merit { double theta, phi, g; };
    auto merit_at = [&](double alpha, double mu_, int with_grad, Merit& out) -> nmpc_status {
        launch_trial_point(M, V, alpha, st);
        launch_model_eval(M, V.yt, nullptr, nullptr, nullptr, V.ct, nullptr, nullptr, nullptr, st);
        launch_merit(M, V, alpha, mu_, o.gamma, with_grad, st);
        h->launches += 3;
        CK(cudaMemcpyAsync(hm, V.scal, 5 * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (with_grad) CK(cudaMemcpyAsync(hm + 5, V.scal + 7, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        out.theta = hm[0]; out.phi = hm[3] > 0.0 ? INFINITY : hm[2] - mu_ * hm[1]; out.g = hm[4];
        return NMPC_OK;
    };
    auto filter_line_search = [&](double mu_) -> nmpc_status {
        Merit k{}, t{};
        TRY(merit_at(0.0, mu_, 1, k));
        const double a_max = hm[5];
        if (!flt_ready) {                                 // [17] Eq. (21): theta_max, theta_min from the starting point
            th_max = o.theta_max_fact * std::max(1.0, k.theta); th_min = o.theta_min_fact * std::max(1.0, k.theta);
            flt_ready = true;
        }
        if (mu_ != flt_mu) { flt.assign(1, {th_max, -INFINITY}); flt_mu = mu_; }       // a new barrier problem: new filter (A-3)
        const double tol = 10.0 * 2.220446049250313e-16 * std::fabs(k.phi);
        double alpha = a_max, accepted = a_max;
        int nback = 0, augment = -1;                      // -1: gave up (reading G20), 0 / 1: accepted without / with augmentation
        for (; nback <= o.ls_max_backtracks; ++nback) {
            TRY(merit_at(alpha, mu_, 0, t));
            bool in_filter = false;
            for (const auto& e : flt) if (t.theta >= e.first && t.phi >= e.second) { in_filter = true; break; }
            const bool switching = k.g < 0.0 && alpha * std::pow(-k.g, o.s_phi) > o.delta_sw * std::pow(k.theta, o.s_theta);
            const bool armijo = t.phi - k.phi - tol <= o.eta_phi * alpha * k.g;
            if (!in_filter) {
                if (k.theta <= th_min && switching) {
                    if (armijo) { accepted = alpha; augment = 0; break; }
                } else if (t.theta <= (1.0 - o.gamma_theta) * k.theta || t.phi - k.phi - tol <= -o.gamma_phi * k.theta) {
                    accepted = alpha; augment = (!switching || !armijo) ? 1 : 0; break;
                }
            }
            alpha *= 0.5;
        }
        if (augment < 0) { accepted = a_max; flt.assign(1, {th_max, -INFINITY}); }
        else if (augment == 1) flt.push_back({(1.0 - o.gamma_theta) * k.theta, k.phi - o.gamma_phi * k.theta});
        last_backtracks = nback;
        hm[7] = accepted;
        CK(cudaMemcpyAsync(V.scal + 7, hm + 7, sizeof(double), cudaMemcpyHostToDevice, st));
        return NMPC_OK;
    };
    auto solve_step_update = [&](double mu_, double tau_) -> nmpc_status {
        pt.begin(&S.ms_solve, 3);                                                 // S8: Eq. (22)-(25)
        TRY(run_newton_solve(h));
        pt.end();
        pt.begin(&S.ms_vector, 4);
        launch_step(M, V, mu_, tau_, nullptr, st); h->launches += 1;                    // S8-S9
        pt.end();
        for (int r = 0; r < o.refine_steps; ++r) {                             // iterative refinement on Eq. (10), first row
            pt.begin(&S.ms_vector, 4);
            launch_refine_residual(M, V, h->eta_cur, h->D.fail_col, st); h->launches++;
            pt.end();
            pt.begin(&S.ms_solve, 3);
            TRY(run_solve(h, V.rho));
            pt.end();
            pt.begin(&S.ms_vector, 4);
            launch_add_correction(M, V, h->D.fail_col, st); launch_step(M, V, mu_, tau_, nullptr, st); h->launches += 2;
            pt.end();
        }
        pt.begin(&S.ms_vector, 4);
        if (o.globalization) TRY(filter_line_search(mu_));                     // Eq. (26): "line search with step size alpha"
        launch_update(M, V, h->D.fail_col, st); h->launches++;                 // S10: Eq. (26)
        pt.end();
        return NMPC_OK;
    };
    while (true) {
        // S2: evaluate c, grad f, J, W (K_SIMD of the paper, Alg. 2 line 5) and the residuals of Eq. (9)
        if (!top_done) {
            pt.begin(&S.ms_eval, 0);
            launch_model_eval(M, V.y, V.wp, V.wm, nullptr, V.c, V.gradf, V.Jval, V.Wval, st); h->launches++;
            pt.end();
            pt.begin(&S.ms_vector, 4);
            launch_residuals(M, V, o.gamma, st); h->launches += 1;
            CK(cudaMemcpyAsync(hs, V.scal, sizeof(double) * 10, cudaMemcpyDeviceToHost, st));
            if (pending) CK(cudaMemcpyAsync(flag, h->D.fail_col, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        }
        top_done = false;
        CK(cudaStreamSynchronize(st));
        pt.end();
        if (pending) {
            pending = false;
            if (*flag != INT_MAX) {                      // the step of iteration it-1 was not taken: redo it with eta > 0
                h->factored = false;
                launch_reset_fail(h->D, st); h->launches += 1;
                double eta = 0.0;
                nmpc_status rs = retry_with_eta(eta);
                if (rs == NMPC_E_INERTIA) { status = rs; goto done; }
                if (rs != NMPC_OK) return rs;
                eta_last = eta;
                TRY(solve_step_update(pend_mu, pend_tau));
                if (trace && it - 1 < trace_cap) trace[it - 1].eta = eta;
                continue;                                // re-evaluate at the new iterate
            }
            h->factored = true; h->eta_cur = 0.0;
        }
        if (it > 0 && trace && it - 1 < trace_cap) { trace[it - 1].alpha_pr = hs[7]; trace[it - 1].alpha_du = hs[8]; }
        if (hs[6] != 0.0) { status = NMPC_E_STEP; break; }
        const double l1 = hs[5];
        const double s_d = std::max(o.s_max, l1 / (double)h->nmult) / o.s_max;
        auto err_mu = [&](double m_) {
            const double comp = std::max(std::fabs(hs[3] - m_), std::fabs(hs[4] - m_));
            return std::max(std::max(hs[0] / s_d, hs[1]), std::max(hs[2], comp / s_d));
        };
        E0 = err_mu(0.0);
        if (E0 <= o.eps_outer) { status = NMPC_OK; break; }                     // S3: Eq. (28)
        if (it >= o.max_iter) { status = NMPC_E_MAXITER; break; }
        double Emu = err_mu(mu);                                               // S4: Eq. (27), barrier update
        while (Emu <= o.kappa_eps * mu && mu > o.eps_outer / 10.0) {
            mu = std::max(o.eps_outer / 10.0, std::min(o.kappa_mu * mu, std::pow(mu, o.theta_mu)));
            Emu = err_mu(mu);
        }
        const double tau = std::max(o.tau_min, 1.0 - mu);                      // S5
        mark_iteration(it);
        if (graph) {                                     // S6-S10 and the next S2 as one graph replay
            double* hp = h->h_pinned + 24;
            hp[0] = mu; hp[1] = tau;
            uint32_t* he = reinterpret_cast<uint32_t*>(hp + 2);  // call numbers: factorization, then 1 + refine_steps solves
            TRY(next_factor_epoch(h, &he[0]));
            for (int r = 0; r <= o.refine_steps; ++r) TRY(next_solve_epochs(h, r == 0 && h->S.aug, &he[1 + 2 * r], &he[2 + 2 * r]));
            CK(cudaGraphLaunch(h->iter_graph, st));
            h->launches += 10 + 4 * o.refine_steps;
            ++nfact;
            pending = true; pend_mu = mu; pend_tau = tau; top_done = true;
            if (trace && it < trace_cap) { trace[it] = nmpc_trace_row{}; trace[it].mu = mu; trace[it].E0 = E0; trace[it].Emu = Emu; }
            ++it;
            continue;
        }
        pt.begin(&S.ms_vector, 4);
        launch_sigma_rhs(M, V, mu, nullptr, st); h->launches += 2;                      // S6
        pt.end();
        pt.begin(&S.ms_assemble, 1);
        launch_assemble_K(M, V.Jval, V.Wval, V.sigx, V.q, 0.0, V.Kval, st); h->launches++;
        pt.end();
        double eta = 0.0;
        ++nfact;
        if (async) {
            uint32_t epoch = 0;
            TRY(next_factor_epoch(h, &epoch));
            launch_factor(h->D, h->F, h->d_Kval, 0.0, epoch, nullptr, st); h->launches += 1;
            h->eta_cur = 0.0;
            pending = true; pend_mu = mu; pend_tau = tau;
        } else {
            pt.begin(&S.ms_factor, 2);
            nmpc_status fs = run_factor(h, 0.0, nullptr);
            pt.end();
            if (fs == NMPC_E_NOT_SPD) {
                nmpc_status rs = retry_with_eta(eta);
                if (rs == NMPC_E_INERTIA) { status = rs; goto done; }
                if (rs != NMPC_OK) return rs;
            } else if (fs != NMPC_OK) return fs;
        }
        if (eta > 0.0) eta_last = eta;
        TRY(solve_step_update(mu, tau));
        if (trace && it < trace_cap) { trace[it] = nmpc_trace_row{}; trace[it].mu = mu; trace[it].E0 = E0; trace[it].Emu = Emu; trace[it].eta = eta; trace[it].backtracks = last_backtracks; }
        ++it;
    }
done:
    // z* is kept for the next warm start (Alg. 1 line 10) only if it is usable: converged, or stopped at max_iter with a finite
    // iterate.  After a non-finite iterate or an exhausted inertia schedule the next solve falls back to the cold start.
    h->have_state = status == NMPC_OK || (status == NMPC_E_MAXITER && hs[6] == 0.0);
    mark_iteration(it);
    launch_objective(M, V, st); h->launches += 1;
    CK(cudaMemcpyAsync(hs + 9, V.scal + 9, sizeof(double), cudaMemcpyDeviceToHost, st));
    if (y_inout) CK(cudaMemcpyAsync(y_inout, V.y, sizeof(double) * M.n, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    S.status = status; S.iters = it; S.factorizations = nfact; S.eta_retries = retries; S.E0 = E0; S.mu = mu; S.eta_last = eta_last;
    S.objective = hs[9];
    for (int k = 0; k < it && k + 1 < n_ev && k < trace_cap; ++k) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->it_ev[k], h->it_ev[k + 1]) == cudaSuccess) trace[k].ms_iter = ms; else cudaGetLastError();
    }
    S.ms_total = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    if (stats) *stats = S;
    return status;
}

// ---- the HyKKT variant of Algorithm 2 (reading G21 of DESIGN.md section 3): same S1..S10 skeleton as
//      nmpc_ipm_solve with the slack rows removed; the direct part is the factorization / solves of K_g, the iterative part a
//      conjugate-gradient loop on the Schur complement whose scalars (two dot products per iteration) are host scalars ----
nmpc_status nmpc_hykkt_solve(nmpc_handle h, int32_t warm, int32_t use_y0, double* y_inout, nmpc_stats* stats, nmpc_trace_row* trace, int32_t trace_cap) {
    if (!h) return NMPC_E_ARG;
    DeviceGuard dg(h);
    if (!h->has_model) { h->err = "nmpc_hykkt_solve needs a model (nmpc_ocp)"; return NMPC_E_STATE; }
    if (h->M.m != h->M.m_dyn) { h->err = "nmpc_hykkt_solve: general rows (nmpc_ocp.n_g) are handled by nmpc_ipm_solve only"; return NMPC_E_STATE; }
    if (use_y0 && !y_inout) return NMPC_E_ARG;
    const nmpc_options& o = h->opt;
    const DevModel& M = h->M;
    const IpmVectors& V = h->V;
    cudaStream_t st = h->stream;
    auto t_begin = std::chrono::steady_clock::now();
    nmpc_stats S{};
    PhaseTimer pt{h, o.time_phases != 0 && stats != nullptr};
    double mu;
    if (warm && h->have_state) {
        launch_warm_push(M, V, o.warm_push, st); h->launches++;
        mu = o.mu_warm;
    } else {
        if (use_y0) CK(cudaMemcpyAsync(V.y, y_inout, sizeof(double) * M.n, cudaMemcpyDeviceToDevice, st));
        launch_cold_init_y(M, V, h->d_uinit, use_y0, o.kappa_push, o.mu0, st);
        launch_fill(M.m, 0.0, V.wp, st);                                       // lam = 0
        h->launches += 2;
        mu = o.mu0;
    }
    launch_fill(M.m, 0.0, V.wm, st);                                           // the model evaluation's lam = w+ - w-
    launch_fill(M.m, o.gamma_h, V.q, st);                                      // J^T diag(q) J = gamma_h J^T J in the assembly
    h->launches += 2;
    const int nmult = h->nmult - (int)M.m;                                     // m equality multipliers + the bound multipliers (no general rows here)
    double eta_last = 0.0, E0 = 0.0;
    int it = 0, nfact = 0, retries = 0;
    int64_t ncg_total = 0;
    nmpc_status status = NMPC_E_MAXITER;
    double* hs = h->h_pinned;
    double* hc = h->h_pinned + 40;                                             // pinned: the two CG dot products
    const int n_ev = trace ? std::min(trace_cap, o.max_iter) + 1 : 0;
    while ((int)h->it_ev.size() < n_ev) { cudaEvent_t e = nullptr; CK(cudaEventCreate(&e)); h->it_ev.push_back(e); }
    auto mark_iteration = [&](int k) {
        if (k < n_ev) cudaEventRecord(h->it_ev[k], st);
        pt.flush(trace && k > 0 && k - 1 < trace_cap ? &trace[k - 1] : nullptr);
    };
    auto kg_solve = [&](double* rhs) -> nmpc_status {                          // Eq. (22)-(25) with the factor of K_g
        pt.begin(&S.ms_solve, 3);
        nmpc_status s = run_solve(h, rhs);
        pt.end();
        return s;
    };
    while (true) {
        pt.begin(&S.ms_eval, 0);
        launch_model_eval(M, V.y, V.wp, V.wm, nullptr, V.c, V.gradf, V.Jval, V.Wval, st); h->launches++;
        pt.end();
        pt.begin(&S.ms_vector, 4);
        launch_hk_residuals(M, V, st); h->launches++;
        CK(cudaMemcpyAsync(hs, V.scal, sizeof(double) * 10, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        pt.end();
        if (it > 0 && trace && it - 1 < trace_cap) { trace[it - 1].alpha_pr = hs[7]; trace[it - 1].alpha_du = hs[8]; }
        if (hs[6] != 0.0) { status = NMPC_E_STEP; break; }
        const double s_d = std::max(o.s_max, hs[5] / (double)nmult) / o.s_max;
        auto err_mu = [&](double m_) {
            const double comp = hs[3] >= hs[4] ? std::max(std::fabs(hs[3] - m_), std::fabs(hs[4] - m_)) : 0.0;   // no bounds: none
            return std::max(std::max(hs[0] / s_d, hs[1]), comp / s_d);
        };
        E0 = err_mu(0.0);
        if (E0 <= o.eps_outer) { status = NMPC_OK; break; }
        if (it >= o.max_iter) { status = NMPC_E_MAXITER; break; }
        double Emu = err_mu(mu);
        while (Emu <= o.kappa_eps * mu && mu > o.eps_outer / 10.0) {
            mu = std::max(o.eps_outer / 10.0, std::min(o.kappa_mu * mu, std::pow(mu, o.theta_mu)));
            Emu = err_mu(mu);
        }
        const double tau = std::max(o.tau_min, 1.0 - mu);
        mark_iteration(it);
        pt.begin(&S.ms_vector, 4);
        launch_hk_rhs(M, V, mu, o.gamma_h, st); h->launches++;                 // Sigma_x, b_g = r1 + gamma_h J^T r2
        pt.end();
        pt.begin(&S.ms_assemble, 1);
        launch_assemble_K(M, V.Jval, V.Wval, V.sigx, V.q, 0.0, V.Kval, st); h->launches++;
        pt.end();
        double eta = 0.0;
        ++nfact;
        pt.begin(&S.ms_factor, 2);
        nmpc_status fs = run_factor(h, 0.0, nullptr);
        pt.end();
        while (fs == NMPC_E_NOT_SPD) {                                         // inertia correction: the schedule of Eq. (13)/(15)
            ++retries;
            if (eta == 0.0) eta = (eta_last == 0.0) ? o.eta_first : std::max(o.eta_min, o.eta_shrink * eta_last);
            else eta = ((eta_last == 0.0) ? o.eta_grow_first : o.eta_grow) * eta;
            if (eta > o.eta_max) { status = NMPC_E_INERTIA; goto done; }
            ++nfact;
            pt.begin(&S.ms_factor, 2);
            fs = run_factor(h, eta, nullptr);
            pt.end();
        }
        if (fs != NMPC_OK) return fs;
        if (eta > 0.0) eta_last = eta;
        // u = K_g^-1 b_g;  CG on S dlam = J u - r2 = J u + c;  dy = K_g^-1 (b_g - J^T dlam)
        pt.begin(&S.ms_solve, 3);
        TRY(run_newton_solve(h));                                              // b_g went through the factorization
        pt.end();
        int ncg = 0;
        {
            double* r = V.r_pp; double* p = V.r_pm; double* Sp = V.t; double* x = V.dwp;
            pt.begin(&S.ms_vector, 4);
            launch_hk_j(M, V, V.dy, V.c, nullptr, r, st);                       // r = J u + c, scal[1] = r . r
            launch_hk_cg_dir(M, 0.0, r, p, x, 1, st); h->launches += 2;         // p = r, x = 0
            CK(cudaMemcpyAsync(hc, V.scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            pt.end();
            double rr = hc[1];
            const double stop = o.cg_tol * o.cg_tol * rr;
            while (ncg < o.cg_max_iter && rr > stop && rr > 0.0) {
                pt.begin(&S.ms_vector, 4);
                launch_hk_jt(M, V, p, nullptr, 1.0, V.rho, st); h->launches++;  // rho = J^T p
                pt.end();
                TRY(kg_solve(V.rho));
                pt.begin(&S.ms_vector, 4);
                launch_hk_j(M, V, V.rho, nullptr, p, Sp, st); h->launches++;    // Sp = J K_g^-1 J^T p, scal[0] = p . Sp
                CK(cudaMemcpyAsync(hc, V.scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                const double a = rr / hc[0];
                launch_hk_cg_update(M, V, a, x, r, p, Sp, st); h->launches++;   // x += a p, r -= a Sp, scal[1] = r . r
                CK(cudaMemcpyAsync(hc, V.scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                const double rr_new = hc[1];
                launch_hk_cg_dir(M, rr_new / rr, r, p, x, 0, st); h->launches++;
                pt.end();
                rr = rr_new;
                ++ncg;
            }
            ncg_total += ncg;
            pt.begin(&S.ms_vector, 4);
            launch_hk_jt(M, V, x, V.b, -1.0, V.dy, st); h->launches++;          // dy <- b_g - J^T dlam
            pt.end();
            TRY(kg_solve(V.dy));
        }
        pt.begin(&S.ms_vector, 4);
        launch_hk_step(M, V, mu, tau, st); launch_hk_update(M, V, st); h->launches += 2;
        pt.end();
        if (trace && it < trace_cap) { trace[it] = nmpc_trace_row{}; trace[it].mu = mu; trace[it].E0 = E0; trace[it].Emu = Emu; trace[it].eta = eta; trace[it].backtracks = ncg; }
        ++it;
    }
done:
    h->have_state = status == NMPC_OK || (status == NMPC_E_MAXITER && hs[6] == 0.0);
    mark_iteration(it);
    launch_objective(M, V, st); h->launches += 1;
    CK(cudaMemcpyAsync(hs + 9, V.scal + 9, sizeof(double), cudaMemcpyDeviceToHost, st));
    if (y_inout) CK(cudaMemcpyAsync(y_inout, V.y, sizeof(double) * M.n, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    S.status = status; S.iters = it; S.factorizations = nfact; S.eta_retries = retries; S.E0 = E0; S.mu = mu; S.eta_last = eta_last;
    S.objective = hs[9];
    for (int k = 0; k < it && k + 1 < n_ev && k < trace_cap; ++k) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->it_ev[k], h->it_ev[k + 1]) == cudaSuccess) trace[k].ms_iter = ms; else cudaGetLastError();
    }
    S.ms_total = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    if (stats) *stats = S;
    return status;
}

nmpc_status nmpc_ipm_solve_batch(nmpc_handle* handles, int32_t count, const int32_t* warm, double* const* y_inout, nmpc_stats* stats) {
    if (!handles || count < 1) return NMPC_E_ARG;
    for (int i = 0; i < count; ++i) {
        if (!handles[i]) return NMPC_E_ARG;
        for (int k = 0; k < i; ++k)
            if (handles[k] == handles[i] || handles[k]->stream == handles[i]->stream) { handles[i]->err = "batch handles must be distinct and own distinct streams"; return NMPC_E_ARG; }
    }
    std::vector<nmpc_status> st((size_t)count, NMPC_OK);
    auto work = [&](int i) { st[i] = nmpc_ipm_solve(handles[i], warm ? warm[i] : 0, 0, y_inout ? y_inout[i] : nullptr, stats ? &stats[i] : nullptr, nullptr, 0); };
    std::vector<std::thread> th;
    th.reserve((size_t)count);
    try { for (int i = 1; i < count; ++i) th.emplace_back(work, i); }
    catch (...) { for (auto& t : th) t.join(); return NMPC_E_ALLOC; }
    work(0);                                              // the calling thread takes the first instance
    for (auto& t : th) t.join();
    for (int i = 0; i < count; ++i) if (st[i] != NMPC_OK) return st[i];
    return NMPC_OK;
}

nmpc_status nmpc_ipm_solve_host(nmpc_handle h, int32_t warm, const double* x0_host, const double* ref_host, double* y_out_host, nmpc_stats* stats) {
    if (!h) return NMPC_E_ARG;
    DeviceGuard dg(h);
    TRY(nmpc_update_params_host(h, x0_host, ref_host));
    nmpc_status st = nmpc_ipm_solve(h, warm, 0, nullptr, stats, nullptr, 0);
    if (y_out_host) {
        double* stage = h->h_pinned + 64 + h->M.desc.nx + (size_t)h->M.desc.N * h->M.desc.nr;
        CK(cudaMemcpyAsync(stage, h->V.y, sizeof(double) * h->M.n, cudaMemcpyDeviceToHost, h->stream));
        CK(cudaStreamSynchronize(h->stream));
        std::memcpy(y_out_host, stage, sizeof(double) * h->M.n);
    }
    return st;
}

}  // extern "C"
