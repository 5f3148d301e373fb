// step.h -- the handle behind the C ABI and the driver of one coarse-graining step (product path).
#pragma once
#include "internal.h"
#include <cmath>
#include <stdexcept>

namespace tatrg {

// DGEMM launches of at least this many flops are the tensor contractions of the path (Eq. 2.18-2.19, 2.9-2.17, A.2-A.11:
// >= 4e9 each at D = 32); the products inside the Cholesky / subspace solvers are <= 3e8.
constexpr double kLargeGemmFlops = 1e9;
constexpr long long kLargePermuteBytes = 100000000;   // permutes of >= 100 MB read + written: larger than L2 (the D^5 tensors at D = 32)

struct Fail {
    int code; std::string msg;
};

}  // namespace tatrg

struct tatrg_ctx {
    double beta = 0, h = 0;
    int D = 0, p = 0;
    uint64_t seed = 0;
    int n_pow = 2, Ktri = 0;
    int Dbond = 0;                   // ILO Triad-ATRG (section 2.3): rank r_bond D of the bond swap and of the decomposition; = D otherwise
    int method = 0;                  // 0: Triad-ATRG, 1: plain ATRG
    bool use_subspace = true;        // leading subspaces by subspace iteration (false: full eigen-decompositions everywhere)
    double tau = tatrg::kTauDefault;
    int timing = 0;
    bool keep_tensors = false;
    bool use_overlap = true;         // TATRG_OPT_OVERLAP: solver chains beside the contractions (saturated steps)
    bool use_graphs = true;          // TATRG_OPT_GRAPHS: replay the iteration steps of the solver chains as CUDA graphs
    int verbose = 0;                 // TATRG_OPT_VERBOSE
    int dgemm_tma = 1;               // TATRG_OPT_DGEMM_TMA
    bool use_cheb = true;            // TATRG_OPT_CHEBYSHEV: Chebyshev-filtered cycles in the subspace iterations of the symmetric (triad) problems
    bool implicit_xy = true;         // TATRG_OPT_IMPLICIT_XY: triad isometries and F, G from U^bond, sigma, V^bond; X, Y never formed (:394)
    bool qr_deficient_hint = false;  // the last QR pre-reduction met numerically rank-deficient operands: the next one goes straight to the rank-revealing path
    tatrg::Pool pool;
    cudaStream_t last_stream = nullptr;
    cudaEvent_t done_ev = nullptr;   // recorded on last_stream after the last step: a call on another stream waits for it first
    tatrg::Tens phi, psi;            // state: Phi[i1,i2,i3,i4,g], Psi[j1,j2,j3,j4,g]
    double* trace_dev = nullptr;     // 1 + 148*8 doubles
    std::vector<double> lnc;         // ln c_j
    int m = 0;
    bool failed = false;
    std::string err;
    std::vector<double> sv_sigma, sv_s;
    double stage_ms[TATRG_NSTAGES] = {0}, stage_flops[TATRG_NSTAGES] = {0};
    double gemm_ms = 0, gemm_flops = 0, perm_ms = 0; long long gemm_calls = 0, perm_calls = 0, perm_bytes = 0;
    double gemm_large_ms = 0, gemm_large_flops = 0; long long gemm_large_calls = 0;   // launches of >= kLargeGemmFlops
    double perm_large_ms = 0; long long perm_large_bytes = 0, perm_large_calls = 0;       // permutes of >= kLargePermuteBytes
    long long last_launches = 0, last_host_syncs = 0;
    tatrg::Counters cnt;
    std::map<std::string, tatrg::Tens> kept;   // tensors of the last step (keep_tensors only)
    std::vector<cudaEvent_t> stage_ev;
    std::vector<cudaGraphExec_t> graveyard;    // replayed graphs of the last step, destroyed at the start of the next one
};

namespace tatrg {
int run_step(tatrg_ctx* c, cudaStream_t st);   // throws nothing; returns status and fills c->err
}
