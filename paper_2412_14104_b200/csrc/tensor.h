// tensor.h -- strided tensor views with named legs and the contraction front end that turns
// "sum over shared legs" into one tensor_gemm launch (gemm.cu).  Host-side index bookkeeping
// only; all arithmetic runs in the kernels.
#pragma once
#include "common.h"

namespace tatrg {

struct Leg {
    char name;
    long long n;
    long long stride;
};

struct Ten {
    double *p = nullptr;
    std::vector<Leg> legs;

    // contiguous row-major tensor, legs named by `names`
    static Ten make(double *p, const char *names, std::initializer_list<long long> dims);
    // same storage, new leg names (same order)
    Ten as(const char *names) const;
    long long size() const
    {
        long long s = 1;
        for (auto &l : legs) s *= l.n;
        return s;
    }
    long long dim(char c) const;
};

// workspace-allocated contiguous tensor
Ten ws_tensor(const char *names, std::initializer_list<long long> dims);

// C (+)= alpha * sum_{legs shared by A and B only} A * B.
// Legs in A, B and C: batch; A and C: rows; B and C: columns.  Any other pattern is an error.
// lower_only: C is a symmetric matrix (rows and columns enumerate the same index in the same order);
// only its lower triangle is guaranteed to be written.
// tri_b: the caller promises that B, as a (summed index) x (column index) matrix in the order of the legs' memory
// strides in A resp. B, vanishes for summed index > column index (a triangular factor applied from the
// right): the k tiles of zeros are skipped.
void contract(const Ten &A, const Ten &B, const Ten &C, double alpha = 1.0, bool accumulate = false,
              bool lower_only = false, bool tri_b = false);

}  // namespace tatrg
