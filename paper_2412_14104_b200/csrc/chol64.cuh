// chol64.cuh -- the 64 x 64 Cholesky factorisation + triangular inverse of one CTA (256 threads), shared by
// chol_block_kernel (chol.cu: diagonal blocks of the blocked factorisation, Cholesky-QR of tall blocks) and the
// fused subspace iteration of the squeezers (sq_iter.cu).  PAPER.md:81-86 Eq. 12; DESIGN.md "Squeezers".
//
// Blocked right-looking elimination of the augmented matrix [S | I] -> [L | L^-1] in four panels of 16 columns.
// The first version eliminated one column per step with all 256 threads (64 steps x one barrier, 320
// instructions per thread and step: 40 - 50 us, the largest single latency of every Cholesky-QR pass); here the
// serial chain of 64 pivots runs inside ONE warp (the 16 x 16 diagonal block and its inverse in registers, columns
// exchanged by shuffles, no barrier), and all threads do the panel and trailing updates as register-tiled
// rank-16 updates from shared memory: three barriers per panel.
#pragma once

namespace tatrg {

constexpr int CH64 = 64;       // block size
constexpr int CH64_NT = 256;   // threads: a 16 x 16 grid, thread (ty, tx) owns the 4 x 4 tile rows 4ty.., columns 4tx..
constexpr int CH64_PB = 16;    // panel width

struct __align__(16) Chol64Work {
    double P[CH64][CH64_PB + 1];       // column block J of S as it stands
    double LpT[CH64_PB][CH64 + 4];     // column block J of L, transposed: LpT[c][i] = L[i][16 J + c] (rows i >= 16 J)
    double WJ[CH64_PB][CH64 + 4];      // row block J of W = (partially eliminated) identity part ...
    double WJn[CH64_PB][CH64 + 4];     // ... and T WJ = row block J of L^-1
    double T[CH64_PB][CH64_PB + 1];    // inverse of the diagonal block of L
};

struct Chol64Smem {
    Chol64Work wk;
    double diag[CH64];
    int bad;
};

// On entry s[a][b] = S[4ty+a][4tx+b] of the SYMMETRISED block (both triangles filled; a block smaller than 64
// padded with the identity), diag[i] = S[i][i], and the CTA has been synchronised after those writes.
// shift_rel > 0 adds shift_rel * max_i S_ii to the first nb diagonal entries.  On exit the lower triangles
// (c <= i) of s and w hold L and L^-1 (entries above the diagonal are to be ignored), diag = diag(L), bad = 1 if a
// pivot was not positive (it is replaced by 1).  Ends with a barrier; wk may be reused by the caller afterwards.
__device__ __forceinline__ void chol64_factor(double (&s)[4][4], double (&w)[4][4], Chol64Work &wk, double *diag, int *bad,
                                              int nb, double shift_rel)
{
    const int t = threadIdx.x, ty = t >> 4, tx = t & 15;
    const int Rt = ty >> 2, Ct = tx >> 2;
    if (t == 0) *bad = 0;
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) w[a][b] = (4 * ty + a == 4 * tx + b) ? 1.0 : 0.0;
    if (shift_rel > 0.0) {
        double mx = 0.0;
        for (int i = 0; i < CH64; ++i) mx = fmax(mx, diag[i]);
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b)
                if (4 * ty + a == 4 * tx + b && 4 * ty + a < nb) s[a][b] += shift_rel * mx;
        __syncthreads();
    }
#pragma unroll 1
    for (int J = 0; J < CH64 / CH64_PB; ++J) {
        const int j0 = CH64_PB * J;
        // (1) the owners publish column block J of S and row block J of W
        if (Ct == J) {
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) wk.P[4 * ty + a][4 * (tx & 3) + b] = s[a][b];
        }
        if (Rt == J) {
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                double2 *o = reinterpret_cast<double2 *>(&wk.WJ[4 * (ty & 3) + a][4 * tx]);
                o[0] = make_double2(w[a][0], w[a][1]);
                o[1] = make_double2(w[a][2], w[a][3]);
            }
        }
        __syncthreads();
        // (2) one warp: D = S[J,J] = L_JJ L_JJ^T and T = L_JJ^-1.  Lane (r, h) holds columns 8h .. 8h+7 of row r.
        // No lane of the warp may take a branch of its own in here: a shuffle issued while the warp is diverged
        // falls back to a lane-by-lane path (BRA.DIV) that costs ~250 cycles per shuffle instead of ~25.
        if (t < 32) {
            const int r = t & 15, h = t >> 4;
            double d[8], tt[8], my_diag = 0.0;
            bool any_bad = false;
            __syncwarp();
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                d[m] = wk.P[j0 + r][8 * h + m];
                tt[m] = (8 * h + m == r) ? 1.0 : 0.0;
            }
#pragma unroll
            for (int k = 0; k < CH64_PB; ++k) {
                constexpr unsigned FULL = 0xffffffffu;
                const int kh = k >> 3, kc = k & 7;
                double piv = __shfl_sync(FULL, d[kc], k + 16 * kh);
                const double colr = __shfl_sync(FULL, d[kc], r + 16 * kh);   // S[r][k]
                const bool ok = piv > 0.0;                     // (false for NaN)
                any_bad = any_bad || !ok;
                piv = ok ? piv : 1.0;
                const double rd = rsqrt(piv), dd = piv * rd;   // one special-function chain instead of sqrt + divide
                my_diag = (r == k) ? dd : my_diag;
                const double lr = (r > k) ? colr * rd : 0.0;
                const double pivcol = d[kc];                   // column k as it stands, before this step's update
#pragma unroll
                for (int m = 0; m < 8; ++m) {
                    const double lcm = __shfl_sync(FULL, pivcol, 8 * h + m + 16 * kh);    // S[8h+m][k]
                    const double wrm = __shfl_sync(FULL, tt[m], k + 16 * h);             // W[k][8h+m]
                    const double l = (8 * h + m > k) ? lcm * rd : 0.0;
                    d[m] = fma(-lr, l, d[m]);
                    const double wv = wrm * rd;
                    tt[m] = (r == k) ? wv : fma(-lr, wv, tt[m]);
                }
                if (h == kh) d[kc] = (r > k) ? lr : (r == k ? dd : 0.0);   // finished column of L
            }
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const bool low = 8 * h + m <= r;
                wk.LpT[8 * h + m][j0 + r] = low ? d[m] : 0.0;
                wk.T[r][8 * h + m] = low ? tt[m] : 0.0;
            }
            if (h == 0) diag[j0 + r] = my_diag;
            if (any_bad && t == 0) *bad = 1;
        }
        __syncthreads();
        // (3) panel: L[i][j0 + c] = sum_m S[i][j0 + m] T[c][m] for the rows below the diagonal block;
        //     row block J of L^-1: WJn = T WJ
        for (int idx = t; idx < (CH64 - j0 - CH64_PB) * CH64_PB; idx += CH64_NT) {
            const int i = j0 + CH64_PB + (idx >> 4), c = idx & 15;
            double sum = 0.0;
#pragma unroll
            for (int m = 0; m < CH64_PB; ++m) sum = fma(wk.P[i][m], wk.T[c][m], sum);
            wk.LpT[c][i] = sum;
        }
#pragma unroll
        for (int n = 0; n < CH64_PB * CH64 / CH64_NT; ++n) {
            const int idx = t + n * CH64_NT, c = idx >> 6, x = idx & 63;
            double sum = 0.0;
#pragma unroll
            for (int m = 0; m < CH64_PB; ++m) sum = fma(wk.T[c][m], wk.WJ[m][x], sum);
            wk.WJn[c][x] = sum;
        }
        __syncthreads();
        // (4) rank-16 updates of the tiles below the panel: S[i][k] -= L[i][J] L[k][J]^T in the trailing block,
        //     W[i][x] -= L[i][J] W[J][x] in the columns filled so far; finished tiles of L and L^-1
        if (Rt > J && Ct <= Rt) {
            auto rank16 = [&](double (&acc)[4][4], const double *second) {
#pragma unroll
                for (int c = 0; c < CH64_PB; ++c) {
                    const double2 *lp = reinterpret_cast<const double2 *>(&wk.LpT[c][4 * ty]);
                    const double2 *sp = reinterpret_cast<const double2 *>(second + c * (CH64 + 4));
                    const double2 l01 = lp[0], l23 = lp[1], x01 = sp[0], x23 = sp[1];
                    const double li[4] = {-l01.x, -l01.y, -l23.x, -l23.y}, xi[4] = {x01.x, x01.y, x23.x, x23.y};
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int b = 0; b < 4; ++b) acc[a][b] = fma(li[a], xi[b], acc[a][b]);
                }
            };
            if (Ct <= J)
                rank16(w, &wk.WJn[0][4 * tx]);
            else
                rank16(s, &wk.LpT[0][4 * tx]);
        }
        if (Ct == J && Rt >= J) {
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) s[a][b] = wk.LpT[4 * (tx & 3) + b][4 * ty + a];
        }
        if (Rt == J) {
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const double2 *o = reinterpret_cast<const double2 *>(&wk.WJn[4 * (ty & 3) + a][4 * tx]);
                const double2 v0 = o[0], v1 = o[1];
                w[a][0] = v0.x;
                w[a][1] = v0.y;
                w[a][2] = v1.x;
                w[a][3] = v1.y;
            }
        }
    }
    __syncthreads();
}

}  // namespace tatrg
