// symbolic.h -- host-once symbolic analysis (step a0; SymCholesky Eq. (18)-(19)).
// Integer work only: ordering P, elimination tree T_elim, column counts, supernode partition S_L, level sets,
// extend-add relative indices, K->panel scatter map, and the J/W/K patterns + J^T Q J gather map of a model.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/nmpc.h"
#include "models.cuh"

namespace nmpc {

// Leading dimension of the column-major r x w panel of a supernode: r rounded up to even, so that every column (and every
// even row offset) is 16-byte aligned for the vector / cp.async loads of the tile kernels.
inline int64_t panel_ld(int64_t r) { return (r + 1) & ~(int64_t)1; }

struct Csr {                       // generic int pattern, row-major
    int64_t nrows = 0, ncols = 0;
    std::vector<int64_t> ptr;
    std::vector<int32_t> idx;
    int64_t nnz() const { return ptr.empty() ? 0 : ptr.back(); }
};

struct ModelMaps {                 // patterns + gather maps of a stage-structured model (empty if no model)
    bool present = false;
    ModelDesc desc{};
    int64_t n = 0, m = 0, m_dyn = 0;   // m = m_dyn dynamics rows (N nx) + the general linear rows
    std::vector<double> g_val;     // values of the general linear rows in J order (J entries from J.ptr[m_dyn] on)
    std::vector<double> cl, cu;    // m: row intervals without the gamma tube: 0 / 0 for the dynamics rows, g_lo / g_hi
    Csr J;                         // m x n, CSR in emission order (sorted columns)
    Csr W;                         // n x n lower CSR
    Csr K;                         // n x n lower CSR: pattern(J^T J) u pattern(W) u diag
    std::vector<int64_t> jt_ptr;   // CSC of J: per column, (J value index, row)
    std::vector<int32_t> jt_idx, jt_row;
    std::vector<int64_t> trip_ptr; // per K entry: triples (ja, jb, row):  K_e += J[ja] q[row] J[jb]
    std::vector<int32_t> trip_a, trip_b, trip_r;
    std::vector<int32_t> k_w;      // per K entry: W value index or -1
    std::vector<int32_t> k_diag;   // per K entry: variable index if diagonal else -1
    std::vector<int32_t> coords;   // n x 3 integer coordinates (stage, i, j) for geometric nested dissection
    std::vector<uint8_t> is_input; // n: 1 for input (u) variables
};

struct Symbolic {
    int64_t n = 0, nnzK = 0;
    Csr K;                              // user (or model) pattern, lower CSR, original indices
    // Right-hand-side row (options.fuse_rhs): the analysed matrix is [K b; b^T 0] with ONE extra variable, index n, ordered
    // last: nt = n + 1 pivot positions, value array [K values (nnzK) | b (n) | 0].  The numeric factorization then leaves
    // v = L^-1 P b (Eq. 22) in the last row of the panels and the forward solve of the Newton system is not run at all.
    // Every array below is over nt pivot positions; the v_* arrays describe the factor of K alone (what the C-ABI reports).
    bool aug = false;
    int64_t nt = 0, nnzKa = 0;
    std::vector<int32_t> v_sn_start, v_rows;
    std::vector<int64_t> v_rows_ptr;
    int64_t v_nnzL = 0, v_panel_doubles = 0, v_update_doubles = 0;
    int32_t v_max_front = 0, v_max_width = 0;
    std::vector<int32_t> perm, iperm;   // perm[new] = old, iperm[old] = new  (Eq. 19)
    std::vector<int32_t> parent;        // elimination tree on pivot positions
    std::vector<int32_t> colcount;      // cc_j incl. diagonal (structure of the un-amalgamated L)
    int32_t ns = 0;
    std::vector<int32_t> sn_start;      // ns+1
    std::vector<int32_t> sn_of_col;     // n
    std::vector<int64_t> rows_ptr;      // ns+1
    std::vector<int32_t> rows;          // per supernode: its w pivot columns then the rows below, increasing
    std::vector<int32_t> sn_parent, sn_level;
    std::vector<int32_t> child_ptr, child_idx;     // children of each supernode, increasing index
    std::vector<int64_t> rel_ptr;       // ns+1 into rel: for supernode s, (r_s - w_s) positions in rows[parent]
    std::vector<int32_t> rel;
    std::vector<int64_t> panel_ptr, upd_ptr;       // ns+1: offsets (doubles) of the panel_ld(r) x w panel / (r-w)^2 update
    std::vector<int64_t> kent_ptr;      // ns+1: K entries landing in each supernode's panel
    std::vector<int32_t> kent_src;      // K value index
    std::vector<int32_t> kent_dst;      // i + j*panel_ld(r) inside the panel
    int32_t nlevels = 0;
    std::vector<int32_t> lvl_ptr, lvl_sn;
    double flops = 0.0;
    int64_t nnzL = 0;
    int32_t max_front = 0, max_width = 0;
    int32_t ordering_used = 0;
    double analyze_ms = 0.0;
    ModelMaps mm;
    std::string error;
};

void default_options(nmpc_options* o);
// Builds J/W/K patterns and gather maps of the model.  Returns false (error set) on a bad description.
bool build_model_maps(const nmpc_ocp* ocp, ModelMaps& mm, std::string& err);
// Full analysis.  pattern may be NULL if ocp names a model.
nmpc_status analyze_symbolic(const nmpc_pattern* pattern, const nmpc_ocp* ocp, const nmpc_options* opt,
                             Symbolic& S, bool augment = false);

}  // namespace nmpc
