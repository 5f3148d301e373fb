// step.h -- the handle behind the C ABI and the driver of one coarse-graining step (product path).
#pragma once
#include "internal.h"
#include <cmath>
#include <stdexcept>

namespace tatrg {

struct Fail {
    int code; std::string msg;
};

}  // namespace tatrg

struct tatrg_ctx {
    double beta = 0, h = 0;
    int D = 0, p = 0;
    uint64_t seed = 0;
    int n_pow = 2, Ktri = 0;
    int method = 0;                  // 0: Triad-ATRG, 1: plain ATRG
    bool use_subspace = true;        // leading subspaces by subspace iteration (false: full eigen-decompositions everywhere)
    double tau = tatrg::kTauDefault;
    int timing = 0;
    bool keep_tensors = false;
    tatrg::Pool pool;
    cudaStream_t last_stream = nullptr;
    tatrg::Tens phi, psi;            // state: Phi[i1,i2,i3,i4,g], Psi[j1,j2,j3,j4,g]
    double* trace_dev = nullptr;     // 1 + 148*8 doubles
    std::vector<double> lnc;         // ln c_j
    int m = 0;
    bool failed = false;
    std::string err;
    std::vector<double> sv_sigma, sv_s;
    double stage_ms[TATRG_NSTAGES] = {0}, stage_flops[TATRG_NSTAGES] = {0};
    double gemm_ms = 0, gemm_flops = 0, perm_ms = 0; long long gemm_calls = 0, perm_calls = 0, perm_bytes = 0;
    long long last_launches = 0;
    tatrg::Counters cnt;
    std::map<std::string, tatrg::Tens> kept;   // tensors of the last step (keep_tensors only)
    std::vector<cudaEvent_t> stage_ev;
};

namespace tatrg {
int run_step(tatrg_ctx* c, cudaStream_t st);   // throws nothing; returns status and fills c->err
}
