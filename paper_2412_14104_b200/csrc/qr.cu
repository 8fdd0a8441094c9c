// qr.cu -- thin QR with R_ii >= 0 ("qr+", reading O9) of a tall row-major matrix,
// as a communication-avoiding Householder TSQR: the "iterations of the QR decomposition in the
// RSVD" of PAPER.md:106 and the canonical form of PAPER.md:37.
//
// Level 0 splits the m rows into blocks of RB rows; every CTA factors its RB x n block with
// Householder reflections in shared memory (robust for rank-deficient blocks: tau = 0), leaves
// the reflectors V in place of the block (stored transposed, [n][rows], so that the apply pass
// reads v_j coalesced) and emits its n x n R.  The stacked R's are the next level's matrix.
// Q is formed top-down: block b of level l applies its reflectors to [C_b; 0], C_b being rows
// [b n, (b+1) n) of the level above; the top starts from diag(sign(R_jj)) so that R_ii >= 0.
#include "ctx.h"

namespace tatrg {

namespace {

constexpr int RB = 256;      // rows per block
constexpr int QR_NT = 256;   // threads per CTA

__device__ __forceinline__ double block_sum256(double v, double *sh)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < QR_NT / 32; ++i) r += sh[i];
    return r;  // all threads
}

// X: rows x n row-major. Block b: rows [b*RB, ...).  Outputs: V^T in place ([n][rb]),
// tau[b*n + j], Rst[b*n*n + i*n + c].
template <int CW>
__global__ void __launch_bounds__(QR_NT) tsqr_factor_kernel(double *__restrict__ X, long long rows, int n,
                                                           double *__restrict__ tau,
                                                           double *__restrict__ Rst)
{
    extern __shared__ double sm[];
    const int ld = n | 1;
    double *S = sm;                 // [RB][ld]
    double *vbuf = S + RB * ld;     // [RB]
    double *red = vbuf + RB;        // [QR_NT/CW][CW]
    double *sc = red + QR_NT;       // scalars + reduction scratch [16]
    constexpr int RG = QR_NT / CW;

    const int t = threadIdx.x;
    const long long r0 = (long long)blockIdx.x * RB;
    const int rb = (int)min((long long)RB, rows - r0);
    double *Xb = X + r0 * n;

    for (int i = t; i < RB * n; i += QR_NT) {
        int r = i / n, c = i - r * n;
        S[r * ld + c] = (r < rb) ? Xb[i] : 0.0;
    }
    __syncthreads();

    const int c = t % CW, rg = t / CW;
    for (int j = 0; j < n; ++j) {
        // (a) norm of the column below the diagonal
        double x = (t > j) ? S[t * ld + j] : 0.0;
        double xn2 = block_sum256(x * x, sc + 4);
        double alpha = S[j * ld + j];
        double beta, tj, scal;
        if (xn2 == 0.0) {
            beta = alpha;
            tj = 0.0;
            scal = 0.0;
        } else {
            beta = -copysign(sqrt(alpha * alpha + xn2), alpha);
            tj = (beta - alpha) / beta;
            scal = 1.0 / (alpha - beta);
        }
        __syncthreads();
        // (c) reflector
        {
            double v = (t > j) ? x * scal : (t == j ? 1.0 : 0.0);
            vbuf[t] = v;
            if (t > j) S[t * ld + j] = v;
            if (t == j) {
                S[j * ld + j] = beta;
                tau[(long long)blockIdx.x * n + j] = tj;
            }
        }
        __syncthreads();
        // (d) w = v^T S[:, j+1:]
        const bool act = (c > j) && (c < n);
        double part = 0.0;
        if (act && tj != 0.0) {
            for (int r = j + ((rg - j) % RG + RG) % RG; r < RB; r += RG) part = fma(vbuf[r], S[r * ld + c], part);
        }
        red[rg * CW + c] = part;
        __syncthreads();
        if (act && tj != 0.0) {
            double w = 0.0;
#pragma unroll
            for (int g = 0; g < RG; ++g) w += red[g * CW + c];
            w *= tj;
            for (int r = j + ((rg - j) % RG + RG) % RG; r < RB; r += RG) S[r * ld + c] = fma(-vbuf[r], w, S[r * ld + c]);
        }
        __syncthreads();
    }
    // R block (upper triangle), then V^T over the block's own storage
    double *Rb = Rst + (long long)blockIdx.x * n * n;
    for (int i = t; i < n * n; i += QR_NT) {
        int r = i / n, cc = i - r * n;
        Rb[i] = (r <= cc) ? S[r * ld + cc] : 0.0;
    }
    for (int i = t; i < n * rb; i += QR_NT) {
        int j = i / rb, r = i - j * rb;
        Xb[i] = (r < j) ? 0.0 : (r == j ? 1.0 : S[r * ld + j]);
    }
}

// Forms Q of one level in place of its V^T blocks.  Cup: the level above (row-major, n columns),
// block b uses rows [b*n, (b+1)*n); if Cup == nullptr the block starts from diag(dsign).
template <int CW>
__global__ void __launch_bounds__(QR_NT) tsqr_apply_kernel(double *__restrict__ X, long long rows, int n,
                                                          const double *__restrict__ tau,
                                                          const double *__restrict__ Cup,
                                                          const double *__restrict__ dsign)
{
    extern __shared__ double sm[];
    const int ld = n | 1;
    double *W = sm;                 // [RB][ld]
    double *vbuf = W + RB * ld;     // [RB]
    double *red = vbuf + RB;        // [RG][CW]
    constexpr int RG = QR_NT / CW;

    const int t = threadIdx.x;
    const long long r0 = (long long)blockIdx.x * RB;
    const int rb = (int)min((long long)RB, rows - r0);
    double *Xb = X + r0 * n;

    for (int i = t; i < RB * n; i += QR_NT) {
        int r = i / n, cc = i - r * n;
        double v = 0.0;
        if (r < n) {
            if (Cup)
                v = Cup[(long long)blockIdx.x * n * n + i];
            else
                v = (r == cc) ? dsign[r] : 0.0;
        }
        W[r * ld + cc] = v;
    }
    const int c = t % CW, rg = t / CW;
    const bool act = c < n;
    for (int j = n - 1; j >= 0; --j) {
        __syncthreads();
        vbuf[t] = (t < rb) ? Xb[(long long)j * rb + t] : 0.0;
        const double tj = tau[(long long)blockIdx.x * n + j];
        __syncthreads();
        if (tj == 0.0) continue;   // uniform across the block
        double part = 0.0;
        if (act)
            for (int r = j + ((rg - j) % RG + RG) % RG; r < RB; r += RG) part = fma(vbuf[r], W[r * ld + c], part);
        red[rg * CW + c] = part;
        __syncthreads();
        if (act) {
            double w = 0.0;
#pragma unroll
            for (int g = 0; g < RG; ++g) w += red[g * CW + c];
            w *= tj;
            for (int r = j + ((rg - j) % RG + RG) % RG; r < RB; r += RG) W[r * ld + c] = fma(-vbuf[r], w, W[r * ld + c]);
        }
    }
    __syncthreads();
    for (int i = t; i < rb * n; i += QR_NT) {
        int r = i / n, cc = i - r * n;
        Xb[i] = W[r * ld + cc];
    }
}

// dsign[j] = R_jj >= 0 ? 1 : -1 ; R <- diag(dsign) R
__global__ void sign_fix_kernel(double *R, int n, double *dsign)
{
    __shared__ double d[128];
    int t = threadIdx.x;
    if (t < n) {
        d[t] = (R[t * n + t] < 0.0) ? -1.0 : 1.0;
        dsign[t] = d[t];
    }
    __syncthreads();
    for (int i = t; i < n * n; i += blockDim.x) R[i] *= d[i / n];
}

size_t smem_for(int n) { return ((size_t)RB * (n | 1) + RB + QR_NT + 16) * sizeof(double); }

template <int CW>
void set_attrs()
{
    static bool done = false;
    if (done) return;
    TATRG_CUDA_CHECK(cudaFuncSetAttribute(tsqr_factor_kernel<CW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)smem_for(CW)));
    TATRG_CUDA_CHECK(cudaFuncSetAttribute(tsqr_apply_kernel<CW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)smem_for(CW)));
    done = true;
}

template <int CW>
void tsqr_impl(double *Y, long long m, int n, double *Rout)
{
    set_attrs<CW>();
    size_t mark = ws_mark();
    struct Level {
        double *X;
        long long rows;
        long long nb;
        double *tau;
        double *Rst;
    };
    std::vector<Level> lv;
    double *X = Y;
    long long rows = m;
    const size_t smem = smem_for(n);
    while (true) {
        Level L;
        L.X = X;
        L.rows = rows;
        L.nb = (rows + RB - 1) / RB;
        L.tau = ws_doubles(L.nb * n);
        L.Rst = ws_doubles(L.nb * n * n);
        tsqr_factor_kernel<CW><<<(unsigned)L.nb, QR_NT, smem, stream()>>>(L.X, L.rows, n, L.tau, L.Rst);
        TATRG_LAUNCH_CHECK();
        count_launch();
        lv.push_back(L);
        if (L.nb == 1) break;
        X = L.Rst;
        rows = L.nb * n;
    }
    double *dsign = ws_doubles(n);
    Level &top = lv.back();
    sign_fix_kernel<<<1, 128, 0, stream()>>>(top.Rst, n, dsign);
    count_launch();
    TATRG_CUDA_CHECK(cudaMemcpyAsync(Rout, top.Rst, sizeof(double) * n * n, cudaMemcpyDeviceToDevice, stream()));
    for (int l = (int)lv.size() - 1; l >= 0; --l) {
        Level &L = lv[l];
        const double *Cup = (l == (int)lv.size() - 1) ? nullptr : lv[l + 1].X;
        tsqr_apply_kernel<CW><<<(unsigned)L.nb, QR_NT, smem, stream()>>>(L.X, L.rows, n, L.tau, Cup, dsign);
        TATRG_LAUNCH_CHECK();
        count_launch();
    }
    ws_release(mark);
}

}  // namespace

// Cholesky-QR2 for a tall, well-conditioned block: C = Y^T Y (tensor-GEMM, split-K), C = L L^T in one
// CTA, Q = Y L^-T (tensor-GEMM), twice; R = L2^T L1^T has a positive diagonal, so this is the same
// unique qr+ factorisation as the Householder route whenever it applies.  It applies when the
// first Cholesky factor exists and its diagonal ratio (a lower bound of cond(Y)) is below 1e5, so
// that cond^2 eps << 1; otherwise nothing has been written and the caller falls back to TSQR.
namespace {

// C (n x n row-major) -> its lower Cholesky factor in place (after adding shift_rel * max
// diag); returns L^-1 as a [d][c] view; mm (optional) receives min / max of diag(L).  Asynchronous.
Ten chol_inv(Ten &C, int n, double shift_rel, int *flag, double *mm)
{
    if (n <= 64) {
        double *Li = ws_doubles(64 * 64);
        chol_block(C.p, n, n, Li, flag, mm, shift_rel);
        Ten L = Ten::make(Li, "dc", {n, 64});
        L.legs[1].n = n;
        return L;
    }
    double *Li = ws_doubles((long long)n * n);
    cholesky_lower_async(C.p, n, shift_rel, Li, flag);
    if (mm) diag_minmax(C.p, n, mm);
    return Ten::make(Li, "dc", {n, n});
}

}  // namespace

bool cholqr2(double *Y, long long m, int n, double *Rout)
{
    size_t mark = ws_mark();
    int *flag = (int *)ws_alloc(sizeof(int));
    double *mm = ws_doubles(2);
    TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    Ten Ym = Ten::make(Y, "rc", {m, n});
    Ten C1 = ws_tensor("cd", {n, n}), C2 = ws_tensor("cd", {n, n});
    contract(Ym, Ym.as("rd"), C1);
    Ten L1i = chol_inv(C1, n, 0.0, flag, mm);   // row d of L^-1; Q[r,d] = sum_c Y[r,c] Linv[d,c]
    struct {
        int f;
        double lo, hi;
    } h;
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h.f, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h.lo, mm, 2 * sizeof(double), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    if (h.f != 0 || !(h.lo > 1e-5 * h.hi)) {
        ws_release(mark);
        return false;
    }
    Ten T = ws_tensor("rd", {m, n});
    contract(Ym, L1i, T);
    contract(T.as("rc"), T, C2);
    Ten L2i = chol_inv(C2, n, 0.0, flag, nullptr);
    contract(T.as("rc"), L2i, Ym.as("rd"));
    // R = L2^T L1^T : R[i][j] = sum_k L2[k][i] L1[j][k]   (C1, C2 now hold L1, L2; upper parts zeroed)
    contract(C2.as("ki"), C1.as("jk"), Ten::make(Rout, "ij", {n, n}));
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h.f, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    ws_release(mark);
    if (h.f != 0) fail(-34, "cholqr2: second Cholesky factorisation failed");
    return true;
}

void cholqr_async(double *Y, long long m, int n, int passes, double shift_rel, int *flag_dev, double *ratio_dev,
                  double *Rout, const double *src, double *last_Linv)
{
    if (n < 1 || n > 256 || passes < 1 || passes > 3) fail(-22, "cholqr_async: n = %d, passes = %d not supported", n, passes);
    if (src == Y) src = nullptr;
    // <= 64 columns: one resident grid (in place)
    if (src && !(n <= 32 && m >= 16384) && n <= 64) {
        TATRG_CUDA_CHECK(cudaMemcpyAsync(Y, src, sizeof(double) * m * n, cudaMemcpyDeviceToDevice, stream()));
        src = nullptr;
    }
    if (cholqr_fused(Y, m, n, passes, shift_rel, flag_dev, ratio_dev, Rout)) {
        if (last_Linv) fill_identity(last_Linv, n);
        return;
    }
    size_t mark = ws_mark();
    Ten Ym = Ten::make(Y, "rc", {m, n});
    Ten T = ws_tensor("rd", {m, n});
    Ten C[3];
    // the applies alternate between Y and T such that the last one lands in Y; with a separate source the first
    // pass reads it directly (no copy of the block); with last_Linv the last factor is handed to the caller
    // instead of being applied (a caller that multiplies Q by a small matrix anyway folds it into that)
    const int applies = last_Linv ? passes - 1 : passes;
    Ten cur = src ? Ten::make(const_cast<double *>(src), "rc", {m, n}) : Ym;
    for (int p = 0; p < passes; ++p) {
        C[p] = ws_tensor("cd", {n, n});
        contract(cur.as("rc"), cur.as("rd"), C[p]);
        Ten Linv = chol_inv(C[p], n, p == 0 ? shift_rel : 0.0, flag_dev, p == 0 ? ratio_dev : nullptr);
        if (p >= applies) {
            TATRG_CUDA_CHECK(cudaMemcpy2DAsync(last_Linv, sizeof(double) * n, Linv.p, sizeof(double) * Linv.legs[0].stride,
                                               sizeof(double) * n, n, cudaMemcpyDeviceToDevice, stream()));
            break;
        }
        Ten nxt = src ? (((applies - 1 - p) & 1) ? T : Ym) : (cur.p == Y ? T : Ym);
        contract(cur.as("rc"), Linv, nxt.as("rd"));       // Q[r,d] = sum_c Y[r,c] Linv[d,c]
        cur = nxt;
    }
    if (cur.p != Y) TATRG_CUDA_CHECK(cudaMemcpyAsync(Y, cur.p, sizeof(double) * m * n, cudaMemcpyDeviceToDevice, stream()));
    if (Rout) {
        // R = L_p^T ... L_1^T (the C[p] now hold the lower factors, upper parts zeroed)
        Ten Rm = Ten::make(Rout, "ij", {n, n});
        if (passes == 1) {
            transpose_small(C[0].p, Rout, n, n);
        } else if (passes == 2) {
            contract(C[1].as("ki"), C[0].as("jk"), Rm);          // R[i][j] = sum_k L2[k][i] L1[j][k]
        } else {
            Ten R12 = ws_tensor("kj", {n, n});
            contract(C[1].as("lk"), C[0].as("jl"), R12);         // (L2^T L1^T)[k][j]
            contract(C[2].as("ki"), R12, Rm);
        }
    }
    ws_release(mark);
}

namespace {

// n > 64: block Gram-Schmidt with reorthogonalisation over two column halves (recursively: tsqr of a
// half wider than 64 columns splits again), each factored by tsqr (the robust route for blocks that are not tall or too ill conditioned for
// Cholesky-QR): Y = [Q1 Q2] [[R11, R12], [0, R22]].
void tsqr_split(double *Y, long long m, int n, double *Rout)
{
    size_t mark = ws_mark();
    const int h1 = n / 2, h2 = n - h1;
    Ten Y1 = ws_tensor("rc", {m, h1}), Y2 = ws_tensor("rd", {m, h2});
    const size_t pitch = sizeof(double) * n;
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Y1.p, sizeof(double) * h1, Y, pitch, sizeof(double) * h1, m, cudaMemcpyDeviceToDevice, stream()));
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Y2.p, sizeof(double) * h2, Y + h1, pitch, sizeof(double) * h2, m, cudaMemcpyDeviceToDevice, stream()));
    Ten R11 = ws_tensor("ce", {h1, h1}), R22 = ws_tensor("df", {h2, h2});
    Ten R12 = ws_tensor("cd", {h1, h2}), Rb = ws_tensor("ed", {h1, h2}), Id = ws_tensor("ce", {h1, h1});
    tsqr(Y1.p, m, h1, R11.p);
    contract(Y1, Y2, R12);                       // R12 = Q1^T Y2
    contract(Y1, R12, Y2, -1.0, true);           // Y2 -= Q1 R12
    contract(Y1.as("re"), Y2, Rb);               // second pass
    contract(Y1.as("re"), Rb, Y2, -1.0, true);
    fill_identity(Id.p, h1);
    contract(Id, Rb, R12, 1.0, true);            // R12 += Rb
    tsqr(Y2.p, m, h2, R22.p);
    {
        // "Twice is enough" holds for the projection of a block of full numerical rank.  When Y is rank
        // deficient (the pair operators of the early steps, r chi above their rank) some columns of the
        // projected Y2 are pure rounding noise, 1e-9 or less of what they were, and the unit vectors tsqr
        // makes of them keep components along Q1 of eps / 1e-9: one more projection AFTER the
        // normalisation, folded into R:  Q2 = Q2'' T + Q1 C  =>  R12 += C R22,  R22 <- T R22.
        Ten Cc = ws_tensor("ed", {h1, h2}), Tm = ws_tensor("gd", {h2, h2}), R22n = ws_tensor("gf", {h2, h2});
        contract(Y1.as("re"), Y2, Cc);
        contract(Y1.as("re"), Cc, Y2, -1.0, true);
        tsqr(Y2.p, m, h2, Tm.p);
        contract(Cc, R22, R12.as("ef"), 1.0, true);
        contract(Tm, R22, R22n);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(R22.p, R22n.p, sizeof(double) * h2 * h2, cudaMemcpyDeviceToDevice, stream()));
    }
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Y, pitch, Y1.p, sizeof(double) * h1, sizeof(double) * h1, m, cudaMemcpyDeviceToDevice, stream()));
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Y + h1, pitch, Y2.p, sizeof(double) * h2, sizeof(double) * h2, m, cudaMemcpyDeviceToDevice, stream()));
    fill_zero(Rout, (long long)n * n);
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Rout, pitch, R11.p, sizeof(double) * h1, sizeof(double) * h1, h1, cudaMemcpyDeviceToDevice, stream()));
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Rout + h1, pitch, R12.p, sizeof(double) * h2, sizeof(double) * h2, h1, cudaMemcpyDeviceToDevice, stream()));
    TATRG_CUDA_CHECK(cudaMemcpy2DAsync(Rout + (long long)h1 * n + h1, pitch, R22.p, sizeof(double) * h2, sizeof(double) * h2, h2, cudaMemcpyDeviceToDevice, stream()));
    ws_release(mark);
}

}  // namespace

void tsqr(double *Y, long long m, int n, double *Rout)
{
    if (n < 1 || m < 1) fail(-22, "tsqr: empty matrix");
    if (n > 256) fail(-22, "tsqr: n = %d > 256 not supported", n);
    if (!(ctx().routes & ROUTE_HOUSEHOLDER_QR) && m >= 16LL * n && m >= 512 && cholqr2(Y, m, n, Rout)) return;
    if (n > 64)
        tsqr_split(Y, m, n, Rout);
    else if (n > 32)
        tsqr_impl<64>(Y, m, n, Rout);
    else if (n > 16)
        tsqr_impl<32>(Y, m, n, Rout);
    else
        tsqr_impl<16>(Y, m, n, Rout);
}

}  // namespace tatrg
