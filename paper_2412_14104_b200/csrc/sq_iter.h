// sq_iter.h -- interface of the fused subspace iteration of a squeezer (sq_iter.cu; caller: step.cpp SqChain)
#pragma once
#include <stddef.h>

namespace tatrg {

constexpr int SQ_UMAX = 16;        // 8-row blocks of the iterate per CTA
constexpr int SQ_MAXSTEPS = 200;   // half steps per launch

// One half step = one byte.  The product is with F (result -> buf[0], operand buf[1]) or, with SQ_TRANS, with
// F^T (read from Ft; result -> buf[1], operand buf[0]); SQ_FROM_START reads the operand from `start` instead.  Then one
// Cholesky-QR pass with the shift `shift` (only the span is carried on), or with SQ_TWO_PASSES two unshifted
// passes (a block that enters a Ritz step).  Bits 3-4: 1 or 2 = min / max of diag(L) of the first pass go to
// ratio[0..1] resp. ratio[2..3].  SQ_WANT_R: the accumulated triangular factor goes to Rout.
enum : unsigned char { SQ_TRANS = 1, SQ_FROM_START = 2, SQ_TWO_PASSES = 4, SQ_RATIO_SHIFT = 3, SQ_WANT_R = 32 };

struct SqIterParams {
    const double *F;       // N2 x N2 row-major
    const double *Ft;      // its transpose (both products read rows)
    const double *start;   // N2 x 64 row-major (SQ_FROM_START)
    double *buf[2];        // N2 x 64 row-major: [0] the iterate on the row side of F, [1] on the column side
    double *Rout;          // 64 x 64 row-major or null
    double *ratio;         // 4 doubles
    int *flag;             // raised (sticky) by a non-positive pivot
    double shift;          // relative diagonal shift of the one-pass steps
    int N2, nsteps;
    unsigned char steps[SQ_MAXSTEPS];
    // set by sq_iter_launch
    double *part, *gram, *Lkeep;
    unsigned *bar;
};

// CTAs of a launch that wants `wanted` of them: every CTA owns 1, 2, 4, 8 or 16 blocks of 8 rows (the smallest
// such count that needs no more than `wanted` CTAs; more than `wanted` only when 16 blocks each are not enough)
int sq_iter_grid(int N2, int wanted);
size_t sq_iter_scratch_doubles(int grid);       // device scratch a launch of `grid` CTAs needs
void sq_iter_launch(SqIterParams p, int wanted, double *scratch);   // asynchronous, on stream(); scratch for sq_iter_grid(N2, wanted)

}  // namespace tatrg
