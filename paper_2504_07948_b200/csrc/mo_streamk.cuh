// mo_streamk.cuh -- the MO contraction V = Phi * C_s as a persistent, warp-specialised, stream-K FP64
// tensor-core GEMM for sm_100a (BASELINE.json north_star item 2).
//
// Why this shape.  The contraction is skinny (M = 5 W rows, N = N_s, K = N_b): 128x128 output tiles give
// 80 CTAs at the 256-water config, 54 % of 148 SMs.  Stream-K instead cuts the flattened (tile, k-block)
// iteration space into 148 equal contiguous ranges, one persistent CTA per SM; a tile whose k-range is
// split over 2-3 CTAs is summed by the CTA that holds its first k-block, in ascending k order
// (deterministic: no atomics), from partial accumulators parked in an L2-resident workspace.
//
// Operand staging.  Both operands live in HBM already in the shape of a shared-memory stage:
//   PhiT [MT][KB][128][36]   (A tile of 128 rows x 32 k, rows padded to 36 doubles)
//   CT   [NT][KB][32][132]   (B tile of 32 k x 128 n, rows padded to 132 doubles)
// so one stage is two contiguous blocks (36,864 B + 33,792 B) that a single producer thread fetches with
// two TMA bulk copies (cp.async.bulk -> SASS UBLKCP) completing on an mbarrier; the row padding makes
// every DMMA fragment load conflict free (a half warp covers 4 rows x 32 B = one 128 B wavefront).
// Eight consumer warps (2 x 4, warp tile 64 x 32 = 32 DMMA m8n8k4 accumulators) never meet a block-wide
// barrier in the main loop: full/empty mbarriers only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gemm_f64.cuh"

namespace qmc {

constexpr int MO_BM = 128, MO_BN = 128, MO_BK = 32;
constexpr int MO_ALD = 36, MO_BLD = 132;
constexpr int MO_A_STAGE = MO_BM * MO_ALD;   // doubles
constexpr int MO_B_STAGE = MO_BK * MO_BLD;   // doubles
#ifndef QMC_MO_STAGES
#define QMC_MO_STAGES 3
#endif
constexpr int MO_STAGES = QMC_MO_STAGES;
constexpr int MO_CONSUMER_WARPS = 8;
// QMC_MO_MERGED (default): no ninth warp -- lane 0 of consumer warp 0 issues the TMA copies between its DMMA steps.  An SM's
// register file is four separate 16K-register files, one per sub-partition, and the warps of a CTA are dealt out to them
// in turn: a ninth warp of 168 registers fills sub-partition 0 (3 x 5376 = 16128), and then no CTA of ANY other kernel
// can become resident on the SM while the contraction runs (measured with a 34-register probe kernel: its CTAs started
// only when the contraction's left).  With eight warps every sub-partition keeps 5632 registers free -- two 64-register
// warps -- which is what the step and basis kernels of the other lane need to run beside the contraction.
#ifndef QMC_MO_MERGED
#define QMC_MO_MERGED 1
#endif
constexpr int MO_THREADS = (MO_CONSUMER_WARPS + (QMC_MO_MERGED ? 0 : 1)) * 32;
constexpr size_t MO_SMEM_BYTES = (size_t)MO_STAGES * (MO_A_STAGE + MO_B_STAGE) * 8 + 2 * MO_STAGES * 8 + 16;
constexpr int MO_TM = 8, MO_TN = 4;  // DMMA tiles per warp (64 x 32)
constexpr int MO_WS_DOUBLES = MO_BM * MO_BN;  // workspace per CTA

__host__ __device__ inline long phiT_index(long row, int f, int KB) {
    return (((row >> 7) * KB + (f >> 5)) * MO_BM + (row & 127)) * MO_ALD + (f & 31);
}
__host__ __device__ inline long cT_index(int l, int j, int KB) {
    return ((((long)(j >> 7)) * KB + (l >> 5)) * MO_BK + (l & 31)) * MO_BLD + (j & 127);
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;\n" ::"n"(MO_CONSUMER_WARPS * 32) : "memory"); }

struct MoArgs {
    const double* PhiT;  // [MT][KB][128][36]
    const double* CT;    // [NT][KB][32][132]
    double* V;           // [M][ldv] row-major
    long ldv;
    int M, N;            // valid rows / columns of V
    int MT, NT, KB;
    double* ws;          // [grid][128*128] partial accumulators
    unsigned* flags;     // [grid] epoch stamps
    unsigned epoch;
    // optional screening plan (MoPlan below): NULL = every k-block of every tile (dense)
    const int* plan_cnt;   // [MT]      kept k-blocks of row tile tm (>= 1)
    const int* plan_pre;   // [MT + 1]  NT * (cnt[0] + ... + cnt[tm-1]); plan_pre[MT] = total iterations
    const int* plan_kb;    // [MT][KB]  the kept k-blocks of tm, ascending
    // optional: [grid][2] %globaltimer (ns) at the start and the end of every CTA -- the span of the launch on the GPU,
    // which CUDA events on the stream cannot give once two lanes run concurrently (an event pair also counts the time the
    // kernel waited for SMs)
    unsigned long long* trace;
};
__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// Where a flattened iteration lies.  Dense: tiles of KB iterations.  Screened: the tiles of row tile tm have cnt[tm]
// iterations each (only the A stages whose largest entry reaches the threshold), tiles ordered tm-major.
struct MoLoc { int tm, tn, i, cnt; long tile_begin; };
template <bool SCREEN>
__device__ __forceinline__ MoLoc mo_locate(const MoArgs& g, long it) {
    MoLoc L;
    if (!SCREEN) {
        const long tile = it / g.KB;
        L.tm = (int)(tile / g.NT); L.tn = (int)(tile - (long)L.tm * g.NT);
        L.cnt = g.KB; L.tile_begin = tile * g.KB; L.i = (int)(it - L.tile_begin);
    } else {
        int tm = 0;
        while (tm + 1 < g.MT && it >= g.plan_pre[tm + 1]) tm++;
        const int c = g.plan_cnt[tm];
        const long r = it - g.plan_pre[tm];
        L.tm = tm; L.tn = (int)(r / c); L.cnt = c; L.i = (int)(r - (long)L.tn * c);
        L.tile_begin = g.plan_pre[tm] + (long)L.tn * c;
    }
    return L;
}

// HALF: 64-row output tiles (the upper or lower half of an A stage; warp tiles 32 x 32) for contractions with so few
// iterations per CTA that 128-row tiles would be split over many CTAs (config 1: 20 tiles x 24 k-blocks on 148 CTAs);
// g.MT then counts 64-row tiles.  Not combined with SCREEN (the plan is per 128-row tile).
template <bool SCREEN, bool HALF>
__global__ void __maxnreg__(168) k_mo_streamk(MoArgs g) {
    static_assert(!(SCREEN && HALF), "screening plans are per 128-row tile");
    constexpr int BM = HALF ? 64 : 128, TM = BM / 16;
    extern __shared__ __align__(128) unsigned char mo_smem_raw[];
    double* stages = reinterpret_cast<double*>(mo_smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(stages + (size_t)MO_STAGES * (MO_A_STAGE + MO_B_STAGE));
    uint64_t* empty = full + MO_STAGES;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < MO_STAGES; s++) { mbar_init(&full[s], 1); mbar_init(&empty[s], MO_CONSUMER_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        if (g.trace) g.trace[2 * blockIdx.x] = global_timer_ns();
    }
    __syncthreads();

    const long total = SCREEN ? (long)g.plan_pre[g.MT] : (long)g.MT * g.NT * g.KB;
    const long it0 = total * blockIdx.x / gridDim.x, it1 = total * (blockIdx.x + 1) / gridDim.x;
    constexpr uint32_t A_BYTES = BM * MO_ALD * 8, STAGE_BYTES = A_BYTES + MO_B_STAGE * 8;

    // ===== producer: one thread streams the stages of this CTA's iteration range.  issue(): the copies of the next
    // iteration, if its stage is free (block: wait for it); returns false when nothing could be issued.  The position in
    // the iteration space advances incrementally (no divisions after the first iteration: with the producer merged into
    // a consumer warp every instruction here is taken from that warp's DMMA stream).
    long p_it = it0;
    uint32_t p_n = 0;
    int p_tm, p_tn, p_i, p_cnt;
    {
        const MoLoc L0 = mo_locate<SCREEN>(g, it0 < it1 ? it0 : 0);
        p_tm = L0.tm; p_tn = L0.tn; p_i = L0.i; p_cnt = L0.cnt;
    }
    auto issue = [&](bool block) -> bool {
        if (p_it >= it1) return false;
        const int s = p_n % MO_STAGES;
        const uint32_t round = p_n / MO_STAGES;
        if (round > 0) {
            if (block) mbar_wait(&empty[s], (round - 1) & 1);
            else if (!mbar_try_wait(&empty[s], (round - 1) & 1)) return false;
        }
        const int kb = SCREEN ? g.plan_kb[(long)p_tm * g.KB + p_i] : p_i;
        double* As = stages + (size_t)s * (MO_A_STAGE + MO_B_STAGE);
        mbar_expect_tx(&full[s], STAGE_BYTES);
        bulk_g2s(As, g.PhiT + ((long)(HALF ? p_tm >> 1 : p_tm) * g.KB + kb) * MO_A_STAGE + (HALF ? (p_tm & 1) * BM * MO_ALD : 0), A_BYTES, &full[s]);
        bulk_g2s(As + MO_A_STAGE, g.CT + ((long)p_tn * g.KB + kb) * MO_B_STAGE, MO_B_STAGE * 8, &full[s]);
        p_it++; p_n++;
        if (++p_i == p_cnt) {   // next tile (tiles are ordered tm-major; a row tile's tiles all have cnt[tm] iterations)
            p_i = 0;
            if (++p_tn == g.NT) {
                p_tn = 0;
                p_tm++;
                if (SCREEN && p_tm < g.MT) p_cnt = g.plan_cnt[p_tm];
            }
        }
        return true;
    };
#if !QMC_MO_MERGED
    if (warp == MO_CONSUMER_WARPS) {
        if (lane == 0)
            while (issue(true)) {
            }
        return;
    }
    constexpr bool merged = false;
#else
    constexpr bool merged = true;
    const bool producer = tid == 0;
    if (producer)
        for (int s = 0; s < MO_STAGES; s++) issue(false);   // the first round needs no wait
#endif

    // ===== consumers =====
    const int wm0 = (warp >> 2) * (BM / 2), wn0 = (warp & 3) * 32;
    const int lr = lane >> 2, lc = lane & 3;
    uint32_t n = 0;
    long it = it0;
    while (it < it1) {
        const MoLoc L = mo_locate<SCREEN>(g, it);
        const int ka = L.i, KBt = L.cnt;  // this segment starts at iteration ka of a tile of KBt iterations
        const long rem = it1 - it;
        const int kb_end = (rem < (long)(KBt - ka)) ? (int)(ka + rem) : KBt;
        const int tm = L.tm, tn = L.tn;
        double acc[TM][MO_TN][2];
#pragma unroll
        for (int i = 0; i < TM; i++)
#pragma unroll
            for (int j = 0; j < MO_TN; j++) acc[i][j][0] = acc[i][j][1] = 0.0;
        for (int kb = ka; kb < kb_end; kb++, n++) {
            const int s = n % MO_STAGES;
            if (merged) {
                // the copies of iteration n must have been issued before anybody can wait for them
                if (tid == 0)
                    while (p_n <= n) issue(true);
                __syncwarp();
            }
            mbar_wait(&full[s], (n / MO_STAGES) & 1);
            const double* As = stages + (size_t)s * (MO_A_STAGE + MO_B_STAGE);
            const double* Bs = As + MO_A_STAGE;
#pragma unroll
            for (int kk = 0; kk < MO_BK / 4; kk++) {
                double af[TM], bf[MO_TN];
#pragma unroll
                for (int i = 0; i < TM; i++) af[i] = As[(wm0 + i * 8 + lr) * MO_ALD + kk * 4 + lc];
#pragma unroll
                for (int j = 0; j < MO_TN; j++) bf[j] = Bs[(kk * 4 + lc) * MO_BLD + wn0 + j * 8 + lr];
#pragma unroll
                for (int i = 0; i < TM; i++)
#pragma unroll
                    for (int j = 0; j < MO_TN; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
                if (merged && (kk & 1) && tid == 0 && p_n < n + MO_STAGES) issue(false);   // refill a stage the moment its last reader has left
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
        it += kb_end - ka;

        // ---- epilogue of this segment
        const bool head = (ka == 0), whole = head && (kb_end == KBt);
        if (!head) {
            // park the partial tile for the owner (CTA with the tile's first k-block), then publish
            double* ws = g.ws + (size_t)blockIdx.x * MO_WS_DOUBLES;
#pragma unroll
            for (int i = 0; i < TM; i++)
#pragma unroll
                for (int j = 0; j < MO_TN; j++) {
                    ws[((i * MO_TN + j) * 2 + 0) * 256 + tid] = acc[i][j][0];
                    ws[((i * MO_TN + j) * 2 + 1) * 256 + tid] = acc[i][j][1];
                }
            __threadfence();
            consumer_bar();
            if (tid == 0) {
                asm volatile("st.release.gpu.global.u32 [%0], %1;\n" ::"l"(g.flags + blockIdx.x), "r"(g.epoch) : "memory");
            }
        } else {
            if (!whole) {
                // owner: add the partials of the CTAs that hold the rest of this tile, in ascending k order
                long covered = L.tile_begin + kb_end;  // first iteration not yet summed
                const long tile_end = L.tile_begin + KBt;
                int peer = blockIdx.x + 1;
                while (covered < tile_end) {
                    const long peer_begin = total * peer / gridDim.x, peer_end = total * (peer + 1) / gridDim.x;
                    if (peer_end > peer_begin) {  // (a CTA whose range is empty never publishes)
                        if (tid == 0) {
                            unsigned v;
                            do {
                                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(g.flags + peer) : "memory");
                                if (v != g.epoch) __nanosleep(64);
                            } while (v != g.epoch);
                        }
                        consumer_bar();
                        const double* ws = g.ws + (size_t)peer * MO_WS_DOUBLES;
#pragma unroll
                        for (int i = 0; i < TM; i++)
#pragma unroll
                            for (int j = 0; j < MO_TN; j++) {
                                acc[i][j][0] += __ldcg(ws + ((i * MO_TN + j) * 2 + 0) * 256 + tid);
                                acc[i][j][1] += __ldcg(ws + ((i * MO_TN + j) * 2 + 1) * 256 + tid);
                            }
                        covered = peer_end < tile_end ? peer_end : tile_end;
                    }
                    peer++;
                }
            }
            const int m0 = tm * BM, n0 = tn * MO_BN;
#pragma unroll
            for (int i = 0; i < TM; i++) {
                const int row = m0 + wm0 + i * 8 + lr;
#pragma unroll
                for (int j = 0; j < MO_TN; j++) {
                    const int col = n0 + wn0 + j * 8 + lc * 2;
                    if (row < g.M && col < g.N) *reinterpret_cast<double2*>(g.V + (long)row * g.ldv + col) = make_double2(acc[i][j][0], acc[i][j][1]);
                }
            }
        }
    }
    if (g.trace && tid == 0) g.trace[2 * blockIdx.x + 1] = global_timer_ns();
}

}  // namespace qmc
