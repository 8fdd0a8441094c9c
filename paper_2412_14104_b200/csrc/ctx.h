// ctx.h -- the one process-global context of libtatrg (state of the renormalised tensor,
// caller-owned workspace, caller-supplied inputs, per-step records).
#pragma once
#include "common.h"
#include "tensor.h"

namespace tatrg {

enum Stage { ST_CANON = 0, ST_SWAP, ST_ISO, ST_TRIAD, ST_GRAM, ST_SQUEEZE, ST_CONTRACT, ST_NORM, ST_COUNT };

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

    Input in[9];
    std::vector<double> spec[10];
    double gaps[4] = {0, 0, 0, 0};

    cudaEvent_t ev[ST_COUNT + 1] = {};
    bool ev_ok = false;
    double stage_ms[ST_COUNT] = {};

    long long launches = 0;
    double flops = 0;
    std::string err;
};

Ctx &ctx();

// step.cpp
void do_init(double beta, double h);
void do_coarse_grain(int direction, int chi, int r, int q, uint64_t seed, int mode);
double do_log_z();
double do_order_parameter(int leg);

}  // namespace tatrg
