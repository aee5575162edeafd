// gemm_f64.cuh -- FP64 tensor-core (DMMA m8n8k4) tile GEMM for sm_100a.
//
// C[b] (op)= A[b] * B[b] for a batch of row-major matrices.  tcgen05 has no FP64 kind, so the FP64
// tensor path on Blackwell is mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4); measured issue rate on B200:
// 37.1 TFLOP/s sustained (profiles/r1_fp64_peak.md), against 33.8 for plain DFMA.
//
// Tiling: CTA tile BM x BN, K step 16, warp tile WM x WN made of 8x8 DMMA tiles, operands staged in
// shared memory by a STAGES-deep cp.async (LDGSTS) ring with +4-double row padding, which makes every
// fragment load conflict free (a half warp touches 4 rows x 32 B = one 128 B wavefront).
// Requirements: K % 16 == 0, N % 2 == 0, lda/ldb/ldc % 2 == 0, 16-byte aligned bases.  M, N may be
// ragged w.r.t. the tile (zero-filled loads, guarded stores).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace qmc {

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to a (kernel, device) pair.  One SmemAttr per kernel (a static at
// its launch site) remembers, per device ordinal, how many bytes have been granted there, so a process that drives several
// GPUs -- or several host threads -- sets the attribute where and when it is needed and nowhere else.  Racing threads at
// worst set the same attribute twice.
// carveout_percent >= 0: the first call on a device also sets the kernel's preferred L1 / shared-memory split (percent of
// the largest shared-memory size).  Only the contraction asks: the step and basis kernels of one lane are meant to share
// an SM with the resident contraction CTA of the other lane, and an SM whose split was sized for the contraction alone
// (the driver's default is the smallest split that fits the running kernel) would have no room for them; the other
// kernels keep the default (asking for the largest split everywhere cost k_step 18 % of its speed: it lives on L1).
struct SmemAttr {
    static constexpr int MAX_DEV = 64;
    std::atomic<size_t> granted[MAX_DEV];   // zero-initialised (static storage): 0 = never configured on that device
    template <class K>
    cudaError_t ensure(K kernel, size_t bytes, int carveout_percent = -1) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        const bool cached = dev >= 0 && dev < MAX_DEV;
        const size_t have = cached ? granted[dev].load(std::memory_order_acquire) : 0;
        const size_t want = bytes > 48 * 1024 ? bytes : 48 * 1024;
        if (have >= want) return cudaSuccess;
        if (have == 0 && carveout_percent >= 0) {
            e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, carveout_percent);
            if (e != cudaSuccess) return e;
        }
        if (bytes > 48 * 1024) {
            e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
            if (e != cudaSuccess) return e;
        }
        if (cached) {
            size_t cur = have;
            while (cur < want && !granted[dev].compare_exchange_weak(cur, want, std::memory_order_release)) {
            }
        }
        return cudaSuccess;
    }
};

template <int BM_, int BN_, int WM_, int WN_, bool BT_, int STAGES_>
struct GemmCfg {
    static constexpr int BM = BM_, BN = BN_, WM = WM_, WN = WN_, STAGES = STAGES_;
    static constexpr bool BT = BT_;  // false: B is K x N row-major; true: B is N x K row-major
    static constexpr int BK = 16;
    static constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN;
    static constexpr int NWARPS = WARPS_M * WARPS_N, NTHREADS = NWARPS * 32;
    static constexpr int TM = WM / 8, TN = WN / 8;  // DMMA tiles per warp
    static constexpr int A_LD = BK + 4;
    static constexpr int B_LD = BT ? (BK + 4) : (BN + 4);
    static constexpr int A_STAGE = BM * A_LD;
    static constexpr int B_STAGE = BT ? BN * B_LD : BK * B_LD;
    static constexpr size_t SMEM_BYTES = (size_t)STAGES * (A_STAGE + B_STAGE) * sizeof(double);
    static_assert(BM % WM == 0 && BN % WN == 0 && WM % 8 == 0 && WN % 8 == 0, "tile shape");
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, bool valid) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 16 : 0;  // src-size 0 -> 16 bytes of zero fill, nothing is read
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem_src), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// Stage one BM x 16 tile of A and one 16 x BN tile of B (k-block kt) into ring slot `slot`.
template <class Cfg>
__device__ __forceinline__ void gemm_load_stage(double* smem, int slot, const double* __restrict__ A, long lda,
                                                const double* __restrict__ B, long ldb, int M, int N, int K, int m0,
                                                int n0, int kt) {
    double* As = smem + (size_t)slot * (Cfg::A_STAGE + Cfg::B_STAGE);
    double* Bs = As + Cfg::A_STAGE;
    const int k0 = kt * Cfg::BK;
    const int tid = threadIdx.x;
    constexpr int ACH = Cfg::BM * (Cfg::BK / 2);
#pragma unroll
    for (int c = tid; c < ACH; c += Cfg::NTHREADS) {
        int row = c >> 3, cc = c & 7;
        int gm = m0 + row;
        bool ok = (gm < M) && (k0 + cc * 2 < K);
        const double* src = ok ? (A + (long)gm * lda + k0 + cc * 2) : A;
        cp_async16(As + row * Cfg::A_LD + cc * 2, src, ok);
    }
    if constexpr (Cfg::BT) {
        constexpr int BCH = Cfg::BN * (Cfg::BK / 2);
#pragma unroll
        for (int c = tid; c < BCH; c += Cfg::NTHREADS) {
            int row = c >> 3, cc = c & 7;
            int gn = n0 + row;
            bool ok = (gn < N) && (k0 + cc * 2 < K);
            const double* src = ok ? (B + (long)gn * ldb + k0 + cc * 2) : B;
            cp_async16(Bs + row * Cfg::B_LD + cc * 2, src, ok);
        }
    } else {
        constexpr int CPR = Cfg::BN / 2;
        constexpr int BCH = Cfg::BK * CPR;
#pragma unroll
        for (int c = tid; c < BCH; c += Cfg::NTHREADS) {
            int row = c / CPR, cc = c % CPR;
            int gk = k0 + row, gn = n0 + cc * 2;
            bool ok = (gk < K) && (gn < N);
            const double* src = ok ? (B + (long)gk * ldb + gn) : B;
            cp_async16(Bs + row * Cfg::B_LD + cc * 2, src, ok);
        }
    }
}

// Accumulate k-blocks [kt_begin, kt_end) of the tile at (m0, n0) into acc (must be initialised).
template <class Cfg>
__device__ __forceinline__ void gemm_mainloop(double (&acc)[Cfg::TM][Cfg::TN][2], double* smem,
                                              const double* __restrict__ A, long lda, const double* __restrict__ B,
                                              long ldb, int M, int N, int K, int m0, int n0, int kt_begin, int kt_end) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wm0 = (warp / Cfg::WARPS_N) * Cfg::WM, wn0 = (warp % Cfg::WARPS_N) * Cfg::WN;
    const int lr = lane >> 2, lc = lane & 3;
    const int nkt = kt_end - kt_begin;
#pragma unroll
    for (int s = 0; s < Cfg::STAGES - 1; s++) {
        if (s < nkt) gemm_load_stage<Cfg>(smem, s, A, lda, B, ldb, M, N, K, m0, n0, kt_begin + s);
        cp_async_commit();
    }
    for (int it = 0; it < nkt; it++) {
        cp_async_wait<Cfg::STAGES - 2>();
        __syncthreads();
        {
            int nxt = it + Cfg::STAGES - 1;
            if (nxt < nkt) gemm_load_stage<Cfg>(smem, nxt % Cfg::STAGES, A, lda, B, ldb, M, N, K, m0, n0, kt_begin + nxt);
            cp_async_commit();
        }
        const double* As = smem + (size_t)(it % Cfg::STAGES) * (Cfg::A_STAGE + Cfg::B_STAGE);
        const double* Bs = As + Cfg::A_STAGE;
#pragma unroll
        for (int kk = 0; kk < Cfg::BK / 4; kk++) {
            double af[Cfg::TM], bf[Cfg::TN];
#pragma unroll
            for (int i = 0; i < Cfg::TM; i++) af[i] = As[(wm0 + i * 8 + lr) * Cfg::A_LD + kk * 4 + lc];
#pragma unroll
            for (int j = 0; j < Cfg::TN; j++) {
                if constexpr (Cfg::BT)
                    bf[j] = Bs[(wn0 + j * 8 + lr) * Cfg::B_LD + kk * 4 + lc];
                else
                    bf[j] = Bs[(kk * 4 + lc) * Cfg::B_LD + wn0 + j * 8 + lr];
            }
#pragma unroll
            for (int i = 0; i < Cfg::TM; i++)
#pragma unroll
                for (int j = 0; j < Cfg::TN; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_async_wait<0>();
    __syncthreads();  // ring may be reused by the caller
}

// Visit the accumulator: f(row, col, v0, v1) with col even, (row, col) and (row, col+1) global indices.
template <class Cfg, class F>
__device__ __forceinline__ void gemm_foreach_acc(double (&acc)[Cfg::TM][Cfg::TN][2], int m0, int n0, F&& f) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wm0 = (warp / Cfg::WARPS_N) * Cfg::WM, wn0 = (warp % Cfg::WARPS_N) * Cfg::WN;
    const int lr = lane >> 2, lc = lane & 3;
#pragma unroll
    for (int i = 0; i < Cfg::TM; i++)
#pragma unroll
        for (int j = 0; j < Cfg::TN; j++) f(m0 + wm0 + i * 8 + lr, n0 + wn0 + j * 8 + lc * 2, acc[i][j][0], acc[i][j][1]);
}

struct GemmArgs {
    const double* A; long lda; long strideA;
    const double* B; long ldb; long strideB;
    double* C; long ldc; long strideC;
    int M, N, K;
};

// Epilogues.  Each has: static constexpr bool preload (true: the accumulators start from the C tile, i.e. the
// kernel computes C += A*B with the C loads issued before the main loop so their latency hides behind the
// operand staging); bool skip(int b) const; void operator()(int b, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const
struct EpiStore {
    static constexpr bool preload = false;
    __device__ bool skip(int) const { return false; }
    __device__ void operator()(int, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row < M && col < N) *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(v0, v1);
    }
};

template <class Cfg, class Epi>
__global__ void __launch_bounds__(Cfg::NTHREADS) gemm_f64_kernel(GemmArgs g, Epi epi) {
    extern __shared__ __align__(16) double gemm_smem[];
    const int b = blockIdx.z;
    if (epi.skip(b)) return;
    const int m0 = blockIdx.y * Cfg::BM, n0 = blockIdx.x * Cfg::BN;
    double acc[Cfg::TM][Cfg::TN][2];
#pragma unroll
    for (int i = 0; i < Cfg::TM; i++)
#pragma unroll
        for (int j = 0; j < Cfg::TN; j++) acc[i][j][0] = acc[i][j][1] = 0.0;
    const double* A = g.A + (long)b * g.strideA;
    const double* B = g.B + (long)b * g.strideB;
    double* C = g.C + (long)b * g.strideC;
    if constexpr (Epi::preload) {
        gemm_foreach_acc<Cfg>(acc, m0, n0, [&](int row, int col, double& v0, double& v1) {
            if (row < g.M && col < g.N) {
                const double2 c = *reinterpret_cast<const double2*>(C + (long)row * g.ldc + col);
                v0 = c.x; v1 = c.y;
            }
        });
    }
    gemm_mainloop<Cfg>(acc, gemm_smem, A, g.lda, B, g.ldb, g.M, g.N, g.K, m0, n0, 0, g.K / Cfg::BK);
    gemm_foreach_acc<Cfg>(acc, m0, n0, [&](int row, int col, double& v0, double& v1) { epi(b, C, g.ldc, g.M, g.N, row, col, v0, v1); });
}

template <class Cfg, class Epi>
cudaError_t gemm_f64_launch(const GemmArgs& g, int batch, const Epi& epi, cudaStream_t st) {
    static SmemAttr attr;
    if (g.K % Cfg::BK != 0) return cudaErrorInvalidValue;  // the main loop runs whole k-blocks: a remainder would be dropped
    cudaError_t e = attr.ensure(gemm_f64_kernel<Cfg, Epi>, Cfg::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    dim3 grid((g.N + Cfg::BN - 1) / Cfg::BN, (g.M + Cfg::BM - 1) / Cfg::BM, batch);
    gemm_f64_kernel<Cfg, Epi><<<grid, Cfg::NTHREADS, Cfg::SMEM_BYTES, st>>>(g, epi);
    return cudaGetLastError();
}

}  // namespace qmc
