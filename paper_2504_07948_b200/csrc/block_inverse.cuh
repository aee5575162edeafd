// block_inverse.cuh -- batched in-place inversion of the Slater matrices at walker creation (set-up, not on the
// per-move path): block Gauss-Jordan with implicit row pivoting, the O(n^3) work done by the FP64 DMMA GEMM.
//
// For block column C_k (NB columns) of every matrix X:
//   k_gjb_panel   one CTA per matrix: LU with partial pivoting on a shared-memory copy of the panel X[unused rows, C_k]
//                 chooses the NB pivot rows R_k (no rows are exchanged: the permutation stays implicit), P = X[R_k, C_k]
//                 is inverted, Fn = -X[:, C_k] (rows of R_k: 0) goes to a side buffer, X[:, C_k] is zeroed;
//                 log|det| += sum log|pivot|, sign *= sign(pivots).
//   k_gjb_rows    T = P^-1 X[R_k, :] with T[:, C_k] = P^-1; rows R_k of X become their final values T.
//   GEMM          X += Fn * T   (rank-NB update of the whole matrix, accumulators preloaded with X)
// After the last block Y = X holds G[i][r(c)] with G X = Pi, Pi[r(c)][c] = 1, so X^-1[c'][r(c)] = Y[r(c')][c]
// (k_gjb_permute), and det X = sign(r) * prod det(P_k).  One Newton-Schulz step (launch_refine_inverse) follows.
#pragma once
#include "device_utils.cuh"
#include "gemm_f64.cuh"

namespace qmc {

constexpr int GJB_NB = 16;       // block width = K of the update GEMM
constexpr int GJB_THREADS = 1024;

struct GjbArgs {
    double* M; long stride; int n, ld;      // matrices (leading n x n block of an ld x ld array, ld % 16 == 0)
    double* Fn;                             // [batch][ld][16]
    double* T;                              // [batch][16][ld]
    double* Pinv;                           // [batch][16][16]
    int* rowof;                             // [batch][ld]   pivot row of column c
    unsigned char* used;                    // [batch][ld]
    double* logdet; int* sign; int* status;
};

// block-wide argmax of (val, idx), lowest index on ties; result broadcast through shared memory
__device__ __forceinline__ void block_argmax(double& val, int& idx, double* redv, int* redi) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, val, o);
        const int oi = __shfl_xor_sync(0xffffffffu, idx, o);
        if (ov > val || (ov == val && oi < idx)) { val = ov; idx = oi; }
    }
    __syncthreads();
    if (lane == 0) { redv[warp] = val; redi[warp] = idx; }
    __syncthreads();
    if (warp == 0) {
        double v = lane < GJB_THREADS / 32 ? redv[lane] : -1.0;
        int i = lane < GJB_THREADS / 32 ? redi[lane] : 0x7fffffff;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, v, o);
            const int oi = __shfl_xor_sync(0xffffffffu, i, o);
            if (ov > v || (ov == v && oi < i)) { v = ov; i = oi; }
        }
        if (lane == 0) { redv[0] = v; redi[0] = i; }
    }
    __syncthreads();
    val = redv[0];
    idx = redi[0];
    __syncthreads();
}

__global__ void __launch_bounds__(GJB_THREADS) k_gjb_panel(GjbArgs g, int k0, int nbk, int nb) {
    extern __shared__ __align__(16) double psm[];
    constexpr int LDQ = GJB_NB + 1;
    const int LDP = nb + 1;  // nb = panel width this matrix size allows in shared memory (16, 8 or 4)
    const int n = g.n, ld = g.ld, b = blockIdx.x, tid = threadIdx.x;
    double* P = psm;                                   // [n][LDP] working copy of the panel
    double* Q = P + (size_t)n * LDP;                   // [16][LDQ] P^-1
    double* redv = Q + GJB_NB * LDQ;                   // [32]
    int* redi = reinterpret_cast<int*>(redv + 32);     // [32]
    int* R = redi + 32;                                // [16]
    unsigned char* U = reinterpret_cast<unsigned char*>(R + GJB_NB);  // [n] 0 free, 1 used by an earlier block, 2 chosen now
    double* M = g.M + (long)b * g.stride;
    unsigned char* used = g.used + (long)b * ld;
    for (int idx = tid; idx < n * nbk; idx += GJB_THREADS) {
        const int i = idx / nbk, j = idx - i * nbk;
        P[i * LDP + j] = M[(long)i * ld + k0 + j];
    }
    for (int i = tid; i < n; i += GJB_THREADS) U[i] = used[i];
    __syncthreads();
    double lad = 0.0;
    int sg = 1;
    for (int j = 0; j < nbk; j++) {
        double best = -1.0;
        int bi = 0x7fffffff;
        for (int i = tid; i < n; i += GJB_THREADS)
            if (U[i] == 0) {
                const double v = fabs(P[i * LDP + j]);
                if (v > best) { best = v; bi = i; }
            }
        block_argmax(best, bi, redv, redi);
        if (!(best > 0.0)) {  // singular (or NaN): flag and stop; the caller checks the status after the last block
            if (tid == 0) g.status[0] = -3;
            return;
        }
        const int r = bi;
        const double piv = P[r * LDP + j];
        if (tid == 0) {
            R[j] = r;
            U[r] = 2;
            lad += log(fabs(piv));
            if (piv < 0.0) sg = -sg;
        }
        __syncthreads();
        const double pinv = 1.0 / piv;
        for (int i = tid; i < n; i += GJB_THREADS)
            if (U[i] == 0) {
                const double f = P[i * LDP + j] * pinv;
                for (int jj = j + 1; jj < nbk; jj++) P[i * LDP + jj] -= f * P[r * LDP + jj];
            }
        __syncthreads();
    }
    // P = X[R, C] (original values) -> Q, inverted in place by Gauss-Jordan in the order R (the order partial pivoting
    // found: no further exchanges needed)
    for (int idx = tid; idx < GJB_NB * LDQ; idx += GJB_THREADS) Q[idx] = 0.0;
    __syncthreads();
    for (int idx = tid; idx < nbk * nbk; idx += GJB_THREADS) {
        const int a = idx / nbk, c = idx - a * nbk;
        Q[a * LDQ + c] = M[(long)R[a] * ld + k0 + c];
    }
    __syncthreads();
    for (int j = 0; j < nbk; j++) {
        const double pv = Q[j * LDQ + j];
        __syncthreads();
        const double pi = 1.0 / pv;
        if (tid < nbk) Q[j * LDQ + tid] = (tid == j ? 1.0 : Q[j * LDQ + tid]) * pi;
        __syncthreads();
        const int a = tid / nbk, c = tid - a * nbk;
        const bool act = tid < nbk * nbk && a != j;
        double nv = 0.0;
        if (act) nv = (c == j ? 0.0 : Q[a * LDQ + c]) - Q[a * LDQ + j] * Q[j * LDQ + c];
        __syncthreads();
        if (act) Q[a * LDQ + c] = nv;
        __syncthreads();
    }
    double* Pg = g.Pinv + (long)b * GJB_NB * GJB_NB;
    for (int idx = tid; idx < GJB_NB * GJB_NB; idx += GJB_THREADS) Pg[idx] = Q[(idx / GJB_NB) * LDQ + (idx % GJB_NB)];
    // Fn = -X[:, C] for the rows outside R (0 for the rows of R and the padding); X[:, C] <- 0 there
    double* Fn = g.Fn + (long)b * ld * GJB_NB;
    for (int idx = tid; idx < ld * GJB_NB; idx += GJB_THREADS) {
        const int i = idx / GJB_NB, a = idx - i * GJB_NB;
        double v = 0.0;
        if (i < n && a < nbk && U[i] != 2) {
            v = -M[(long)i * ld + k0 + a];
            M[(long)i * ld + k0 + a] = 0.0;
        }
        Fn[idx] = v;
    }
    if (tid < nbk) {
        used[R[tid]] = 1;
        g.rowof[(long)b * ld + k0 + tid] = R[tid];
    }
    if (tid == 0) {
        g.logdet[b] += lad;
        g.sign[b] *= sg;
    }
}

// T = P^-1 X[R, :] (columns of C: P^-1 itself); rows R of X take their final values.  One thread per column.
__global__ void __launch_bounds__(256) k_gjb_rows(GjbArgs g, int k0, int nbk) {
    __shared__ double Q[GJB_NB * GJB_NB];
    __shared__ int R[GJB_NB];
    const int b = blockIdx.y, c = blockIdx.x * 256 + threadIdx.x, ld = g.ld;
    Q[threadIdx.x] = g.Pinv[(long)b * GJB_NB * GJB_NB + threadIdx.x];
    if (threadIdx.x < nbk) R[threadIdx.x] = g.rowof[(long)b * ld + k0 + threadIdx.x];
    __syncthreads();
    if (c >= ld) return;
    double* M = g.M + (long)b * g.stride;
    double* T = g.T + (long)b * GJB_NB * ld;
    double t[GJB_NB];
#pragma unroll
    for (int a = 0; a < GJB_NB; a++) t[a] = 0.0;
    if (c < g.n) {
        if (c >= k0 && c < k0 + nbk) {
#pragma unroll
            for (int a = 0; a < GJB_NB; a++) t[a] = Q[a * GJB_NB + (c - k0)];
        } else {
            for (int q = 0; q < nbk; q++) {
                const double x = M[(long)R[q] * ld + c];
#pragma unroll
                for (int a = 0; a < GJB_NB; a++) t[a] += Q[a * GJB_NB + q] * x;
            }
        }
        for (int a = 0; a < nbk; a++) M[(long)R[a] * ld + c] = t[a];
    }
#pragma unroll
    for (int a = 0; a < GJB_NB; a++) T[(long)a * ld + c] = t[a];
}

// X^-1[c'][r(c)] = Y[r(c')][c]
__global__ void __launch_bounds__(256) k_gjb_permute(GjbArgs g, double* __restrict__ out) {
    const int b = blockIdx.z, cp = blockIdx.y, c = blockIdx.x * 256 + threadIdx.x;
    if (c >= g.n) return;
    const int* rowof = g.rowof + (long)b * g.ld;
    const double* M = g.M + (long)b * g.stride;
    out[(long)b * g.stride + (long)cp * g.ld + rowof[c]] = M[(long)rowof[cp] * g.ld + c];
}
__global__ void __launch_bounds__(256) k_gjb_copy_back(GjbArgs g, const double* __restrict__ in) {
    const int b = blockIdx.z, r = blockIdx.y, c = blockIdx.x * 256 + threadIdx.x;
    if (c >= g.n) return;
    g.M[(long)b * g.stride + (long)r * g.ld + c] = in[(long)b * g.stride + (long)r * g.ld + c];
}
// sign of the permutation c -> r(c) by cycle counting (one thread per matrix)
__global__ void k_gjb_perm_sign(GjbArgs g, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const int* rowof = g.rowof + (long)b * g.ld;
    unsigned char* seen = g.used + (long)b * g.ld;  // all 1 after the last block: reuse as "not yet visited"
    int sg = 1;
    for (int c = 0; c < g.n; c++) {
        if (seen[c] != 1) continue;
        int len = 0;
        for (int x = c; seen[x] == 1; x = rowof[x]) { seen[x] = 3; len++; }
        if ((len & 1) == 0) sg = -sg;
    }
    g.sign[b] *= sg;
}

inline int gjb_panel_width(int n) {
    for (int nb = GJB_NB; nb > 1; nb >>= 1)
        if ((size_t)n * (nb + 1) * 8 + 8192 + n <= 200 * 1024) return nb;
    return 0;
}
inline size_t gjb_panel_smem(int n, int nb) { return (size_t)n * (nb + 1) * 8 + GJB_NB * (GJB_NB + 1) * 8 + 32 * 8 + 32 * 4 + GJB_NB * 4 + n + 64; }

struct EpiAccum {  // C += A*B, accumulators preloaded from C
    static constexpr bool preload = true;
    __device__ bool skip(int) const { return false; }
    __device__ void operator()(int, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row < M && col < N) *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(v0, v1);
    }
};

}  // namespace qmc
