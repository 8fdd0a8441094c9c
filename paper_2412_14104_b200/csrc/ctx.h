// ctx.h -- the one process-global context of libtatrg (state of the renormalised tensor,
// caller-owned workspace, caller-supplied inputs, per-step records).
#pragma once
#include "common.h"
#include "tensor.h"

namespace tatrg {

enum Stage { ST_CANON = 0, ST_SWAP, ST_ISO, ST_TRIAD, ST_GRAM, ST_SQUEEZE, ST_CONTRACT, ST_NORM, ST_COUNT };

// tatrg_set_routes: forces the robust routes of the step (for tests: fast and robust routes must agree)
enum Route { ROUTE_PLAIN_SWAP = 1, ROUTE_HOUSEHOLDER_QR = 2, ROUTE_DENSE_SQUEEZER = 4, ROUTE_SEQUENTIAL_ISO = 8, ROUTE_TMA_PRODUCER = 16,
             ROUTE_UNFUSED_SQUEEZER = 32 };

struct Input {
    const double *ptr = nullptr;
    size_t n = 0;
    int on_device = 0;
};

struct Ctx {
    cudaStream_t stream = nullptr;
    char *ws = nullptr;
    size_t ws_bytes = 0;
    size_t lo = 0, hi = 0;  // scratch = [lo, hi)
    size_t peak = 0;

    bool inited = false;
    double beta = 0, h = 0;
    int dims[4] = {0, 0, 0, 0};
    int bond = 0;
    int step = 0;
    double log_acc = 0;
    double *phi = nullptr, *psi = nullptr;  // [d1,d2,d3,d4,bond] row-major, inside ws
    bool state_low = true;                  // the state sits at the low end of ws
    size_t state_bytes = 0;

    // independent chains of small kernels (the three squeezers, the four isometries) run on side
    // streams forked from / joined to `stream` with events; each chain bump-allocates from its own
    // slice of the free workspace (step.cpp: Fork)
    static constexpr int MAX_CHAINS = 8;
    cudaStream_t side[MAX_CHAINS] = {};
    cudaEvent_t fork_ev = nullptr, join_ev[MAX_CHAINS] = {}, dep_ev[MAX_CHAINS] = {};
    bool side_ok = false;
    char *pinned = nullptr;                 // page-locked host scratch for asynchronous read-backs
    static constexpr size_t PINNED_BYTES = 1 << 16;

    // host-resident inputs of a step are uploaded by a copy stream from the start of the step on
    // (step.cpp: prefetch_inputs), overlapping the canonical form; get_input waits for the event
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t pre_ev[9] = {};
    cudaEvent_t pre_t0 = nullptr, pre_t1 = nullptr;   // timing events around the step's uploads
    bool pre_timed = false;
    double h2d_ms = 0;                                // copy-stream time of the last step's uploads
    size_t h2d_bytes = 0;
    double *pre[9] = {};
    size_t pre_n[9] = {};

    Input in[9];
    int sq_hist[4][3] = {};                 // subspace iterations each squeezer needed, per direction (step.cpp: SqChain)
    int sm_reserve = 0;                     // SMs the persistent GEMM leaves to concurrent chains (step.cpp)
    int chol_ctas = 16;                     // CTAs of the resident blocked Cholesky (chol.cu); 0: one launch per panel step
    int routes = 0;                         // mask of Route: robust routes forced by tatrg_set_routes
    // Phi / Psi split over two GPUs (tatrg_set_side_split): the halves of the contraction this process
    // computes (bit 0 Phi, bit 1 Psi) and the caller's exchange that completes the other half before the normalisation
    int side_mask = 3;
    int (*exchange)(void *user, double *phi, double *psi, long long n, void *stream) = nullptr;
    void *exchange_user = nullptr;
    bool keep_iso = false;                  // tatrg_keep_isometries: host copies of U^A, U^X, U^Y, U^D of the last step
    std::vector<double> iso[4];
    int iso_rows = 0, iso_cols = 0;
    std::vector<double> iso_H[4];           // wide isometries: Ritz matrices whose spectra are computed on demand
    bool iso_pending[4] = {false, false, false, false};
    std::vector<double> spec[10];
    double gaps[4] = {0, 0, 0, 0};

    cudaEvent_t ev[ST_COUNT + 1] = {};
    bool ev_ok = false;
    double stage_ms[ST_COUNT] = {};
    double host_t[ST_COUNT + 1] = {};       // host clock at the stage marks (trace)

    long long launches = 0;
    double flops = 0;
    std::string err;

    // optional per-launch timing of the tensor-GEMM kernel (tatrg_set_profile): CUDA event pairs
    // around every tgemm launch of a step, summed per stage when the step ends
    int prof = 0;   // 0 off, 1 the 128x128 tile only, 2 every tensor-GEMM launch
    int cur_stage = 0;
    std::vector<cudaEvent_t> prof_ev;   // pool, two per launch
    struct ProfRec {
        int stage;
        int big;
        double flops;
        int shape[5];   // M, N, K, batch, ksplit
    };
    int prof_shape[5] = {0, 0, 0, 0, 0};
    std::vector<std::pair<std::string, cudaEvent_t>> tmarks;   // TATRG_TRACE: labelled events inside a step
    double host_contract_s = 0;   // host seconds spent inside contract() (trace only)
    long long host_contract_n = 0;
    std::vector<ProfRec> prof_rec;
    double gemm_ms[ST_COUNT][2] = {};      // [stage][0: 64x64 tile, 1: 128x128 tile]
    double gemm_fl[ST_COUNT][2] = {};
    long long gemm_n[ST_COUNT][2] = {};
};

Ctx &ctx();

// step.cpp
void do_init(double beta, double h);
void do_coarse_grain(int direction, int chi, int r, int q, uint64_t seed, int mode);
double do_log_z();
double do_order_parameter(int leg);
void resolve_iso_spectra();
// api.cpp : per-launch GEMM timing
int prof_begin(double flops, int big);   // returns slot or -1
void prof_end(int slot);
void prof_collect();                     // after a stream sync: fold the event pairs into gemm_ms

}  // namespace tatrg
