// window_kernel.cuh -- the mid-size path (row f4, upper half; the paper's own 82-240-electron molecules, PAPER.md L265,
// L279-302, and configs[1]): ONE launch moves the walkers through a whole delay window -- k consecutive electrons --
// instead of three launches per electron.
//
// At 33..256 electrons per spin the per-electron kernels are short (13-32 us) and each runs far below its roofline: the
// contraction of configs[1] is 0.5 GFLOP cut into 480 (tile, k-block) iterations for 148 CTAs, so its time is fill, drain
// and the stream-K fix-up.  Here a CTA owns G = 4 walkers for the whole window and does, per electron, everything the
// three kernels did, without leaving the SM:
//   [A] accept/reject + commit of electron p-1 and proposal of electron p: the body of k_step (step_kernel.cuh), one
//       128-thread group per walker, the four groups side by side on named barriers;
//   [B] the basis functions at the G proposed positions, straight into shared memory as the A operand (5 G rows x N_b);
//       they never reach HBM ("FP64 ALU if fused into the GEMM producer");
//   [C] the MO rows V = Phi C_s on FP64 DMMA tiles, the coefficient tiles (the pre-tiled CT of the large path) streamed
//       from L2 by TMA bulk copies through a 2-stage mbarrier ring; V goes to global memory (L2) where [A] reads it.
// Walkers are independent, so nothing is ever synchronised across CTAs.  The delayed-update window (Vbuf, Wbuf, S^-1) is
// the one of the large path, in global memory; the flush between two windows is the large path's batched DMMA GEMMs.
#pragma once
#include "step_kernel.cuh"

namespace qmc {

constexpr int WIN_G = 4;                 // walkers per CTA
constexpr int WIN_GT = 128;              // threads per walker group
constexpr int WIN_THREADS = WIN_G * WIN_GT;
constexpr int WIN_MMA_WARPS = 8;         // warps 0..7 contract; warp 8 lane 0 streams the coefficient stages
constexpr int WIN_STAGES = 4;             // ring of HALF coefficient blocks (16 of the 32 k-rows of a CT block, 16.9 KB each)
constexpr int WIN_HALF = MO_B_STAGE / 2;  // doubles per ring slot
constexpr int WIN_MT = (5 * WIN_G + 7) / 8;   // 8-row DMMA tiles over the 5 G rows

struct WinLayout {
    int step, phi_ld, phi, cst, bars, total;   // offsets in doubles
    __host__ __device__ WinLayout(int nsp, int kp, int nbp) {
        step = 0;
        const int per_group = (StepLayout(nsp, kp, WIN_GT / 32).total + 1) & ~1;
        phi_ld = nbp + 4;                       // row stride = 32 B mod 128 B: conflict-free DMMA fragment loads
        phi = step + WIN_G * per_group;
        cst = phi + 5 * WIN_G * phi_ld;
        cst = (cst + 15) & ~15;                 // 128-byte alignment of the TMA destination
        bars = cst + WIN_STAGES * WIN_HALF;
        total = bars + 2 * WIN_STAGES + 2;   // full[], empty[], phi_hi
    }
};
inline size_t window_smem_bytes(int nsp, int kp, int nbp) { return (size_t)WinLayout(nsp, kp, nbp).total * sizeof(double); }

struct WinArgs {
    int spin, p_first, n_steps;   // electrons p_first .. p_first + n_steps - 1 of this spin (one delay window)
    long log_base;                // (sweep index in the log) * n_e * W_total
    int W_total;                  // walkers of the whole crowd (stride of a log row)
    uint32_t step;
    double tau, sqrt_tau;
};

// value / gradient / Laplacian of the functions of one shell at one point, handed to emit(m, v[5]) (formulas: k_basis)
template <class Emit>
__device__ __forceinline__ void win_eval_shell(const SysDev& s, const KbShell& rec, double px, double py, double pz, Emit&& emit) {
    const double x = px - rec.x, y = py - rec.y, z = pz - rec.z;
    const double t = x * x + y * y + z * z;
    const Exp3 ex = exp_neg3(-rec.a[0] * t, -rec.a[1] * t, -rec.a[2] * t);
    const double e0 = rec.c[0] * ex.a, e1 = rec.c[1] * ex.b, e2 = rec.c[2] * ex.c;
    double g = e0, g1 = -(rec.a[0] * e0), g2 = rec.a[0] * rec.a[0] * e0;
    g += e1; g1 -= rec.a[1] * e1; g2 += rec.a[1] * rec.a[1] * e1;
    g += e2; g1 -= rec.a[2] * e2; g2 += rec.a[2] * rec.a[2] * e2;
    for (int p = 3; p < rec.nprim; p++) {
        const double al = __ldg(s.alpha + rec.poff + p);
        const double e = __ldg(s.coef + rec.poff + p) * exp(-al * t);
        g += e; g1 -= al * e; g2 += al * al * e;
    }
    const double lapfac = (double)(4 * rec.l + 6) * g1 + 4.0 * t * g2;
    const double tg1 = 2.0 * g1;
    auto fn = [&](int m, double S, double Sx, double Sy, double Sz) {
        const double v[5] = {S * g, g * Sx + tg1 * S * x, g * Sy + tg1 * S * y, g * Sz + tg1 * S * z, S * lapfac};
        emit(m, v);
    };
    const double s3 = 1.7320508075688772;
    if (rec.l == 0) {
        fn(0, 1.0, 0.0, 0.0, 0.0);
    } else if (rec.l == 1) {
        fn(0, x, 1.0, 0.0, 0.0);
        fn(1, y, 0.0, 1.0, 0.0);
        fn(2, z, 0.0, 0.0, 1.0);
    } else {
        fn(0, s3 * x * y, s3 * y, s3 * x, 0.0);
        fn(1, s3 * y * z, 0.0, s3 * z, s3 * y);
        fn(2, z * z - 0.5 * (x * x + y * y), -x, -y, 2.0 * z);
        fn(3, s3 * x * z, s3 * z, 0.0, s3 * x);
        fn(4, (0.5 * s3) * (x * x - y * y), s3 * x, -s3 * y, 0.0);
    }
}

__global__ void __launch_bounds__(WIN_THREADS, 1) k_window(SysDev s, WalkDev wd, WinArgs a) {
    extern __shared__ __align__(128) double wsm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grp = tid / WIN_GT, gtid = tid - grp * WIN_GT;
    const int spin = a.spin, nsp = s.nsp[spin], kp = wd.kp, nbp = s.nbp, KB = s.kb, NT = s.nt[spin];
    const WinLayout L(nsp, kp, nbp);
    const int per_group = (StepLayout(nsp, kp, WIN_GT / 32).total + 1) & ~1;
    double* sm_g = wsm + L.step + grp * per_group;
    double* phi = wsm + L.phi;
    double* cst = wsm + L.cst;
    uint64_t* full = reinterpret_cast<uint64_t*>(wsm + L.bars);
    uint64_t* empty = full + WIN_STAGES;
    uint64_t* phi_hi = empty + WIN_STAGES;
    const int kbh = (KB + 1) / 2;
    const int w0 = blockIdx.x * WIN_G;
    const int w = w0 + grp;
    const bool live = w < wd.W;
    const int n_live = wd.W - w0 < WIN_G ? wd.W - w0 : WIN_G;   // walkers of this CTA
    const int rows = 5 * n_live;
    const GroupSync<WIN_GT> gsync{1 + grp};
    const int e0 = spin == 0 ? 0 : s.ns[0];

    if (tid == 0) {
        for (int st = 0; st < WIN_STAGES; st++) { mbar_init(&full[st], 1); mbar_init(&empty[st], WIN_MMA_WARPS); }
        mbar_init(phi_hi, WIN_THREADS / 32 - WIN_MMA_WARPS - 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    // padded functions (n_basis .. nbp) are never written: zero the operand once
    for (int i = tid; i < 5 * WIN_G * L.phi_ld; i += WIN_THREADS) phi[i] = 0.0;
    __syncthreads();

    uint32_t n_load = 0, n_use = 0;   // stages issued (producer thread) / consumed (MMA warps) since the start of the kernel
    for (int i = 0; i <= a.n_steps; i++) {
        const int p_prop = i < a.n_steps ? a.p_first + i : -1;
        const int p_acc = i > 0 ? a.p_first + i - 1 : -1;
        // ---- [A] accept p_acc, propose p_prop: one group per walker
        if (live) {
            const long log_off = a.log_base + (long)(e0 + (p_acc >= 0 ? p_acc : 0)) * a.W_total;
            step_body<WIN_GT, true>(s, wd, w, gtid, sm_g, gsync, spin, p_acc, p_prop, log_off, a.step, a.tau, a.sqrt_tau, 1);
        }
        if (p_prop < 0) break;
        __syncthreads();   // the proposals (wd.rp) are written
        // ---- [B] basis functions at the proposed positions -> phi[row = g*5 + c][function].  The shells of the lower half of
        // K by all warps; those of the upper half by warps 9..15 while warps 0..7 already contract the lower half (they
        // wait at `phi_hi` before they enter the upper half).
        auto basis_items = [&](int it0, int it1, int t0, int nt) {
            for (int it = it0 + t0; it < it1; it += nt) {
                const int idx = it / n_live, g = it - idx * n_live;
                const int ks = __ldg(s.win_items + idx);
                const int kb = ks >> 5;
                KbShell rec;
                {
                    const double2* src = reinterpret_cast<const double2*>(s.kb_list + ks);
                    double2* dst = reinterpret_cast<double2*>(&rec);
#pragma unroll
                    for (int q = 0; q < 6; q++) dst[q] = __ldg(src + q);
                }
                const double* r3 = wd.rp + 3 * (size_t)(w0 + g);
                const int c0 = rec.f0 - kb * 32;
                double* base = phi + (size_t)(g * 5) * L.phi_ld + kb * 32;
                win_eval_shell(s, rec, r3[0], r3[1], r3[2], [&](int m, const double (&v)[5]) {
                    const int c = c0 + m;
                    if (c < 0 || c >= 32) return;   // the part of a straddling shell that belongs to the neighbour block
#pragma unroll
                    for (int q = 0; q < 5; q++) base[q * L.phi_ld + c] = v[q];
                });
            }
        };
        basis_items(0, s.n_win_first * n_live, tid, WIN_THREADS);
        __syncthreads();
        // ---- [C] V = Phi C: warps 0..7 contract (each 16 columns of a 128-column tile), warp 8 lane 0 streams C
        if (warp == WIN_MMA_WARPS) {
            if (lane == 0) {
                for (int tn = 0; tn < NT; tn++)
                    for (int hb = 0; hb < 2 * KB; hb++, n_load++) {   // half blocks are contiguous in CT: 16 rows of 132
                        const int st = n_load % WIN_STAGES;
                        const uint32_t round = n_load / WIN_STAGES;
                        if (round > 0) mbar_wait(&empty[st], (round - 1) & 1);
                        mbar_expect_tx(&full[st], WIN_HALF * 8);
                        bulk_g2s(cst + (size_t)st * WIN_HALF, s.CT[spin] + (long)tn * KB * MO_B_STAGE + (long)hb * WIN_HALF, WIN_HALF * 8, &full[st]);
                    }
            }
        } else if (warp > WIN_MMA_WARPS) {
            basis_items(s.n_win_first * n_live, s.n_win_items * n_live, tid - (WIN_MMA_WARPS + 1) * 32, WIN_THREADS - (WIN_MMA_WARPS + 1) * 32);
            __syncwarp();
            if (lane == 0) mbar_arrive(phi_hi);
        }
        if (warp < WIN_MMA_WARPS) {
            const int lr = lane >> 2, lc = lane & 3;
            const int wn0 = warp * 16;
            for (int tn = 0; tn < NT; tn++) {
                double acc[WIN_MT][2][2];
#pragma unroll
                for (int mi = 0; mi < WIN_MT; mi++)
#pragma unroll
                    for (int j = 0; j < 2; j++) acc[mi][j][0] = acc[mi][j][1] = 0.0;
                for (int hb = 0; hb < 2 * KB; hb++, n_use++) {
                    if (tn == 0 && hb == 2 * kbh) mbar_wait(phi_hi, i & 1);   // the upper half of the operand is complete
                    const int st = n_use % WIN_STAGES;
                    mbar_wait(&full[st], (n_use / WIN_STAGES) & 1);
                    const double* Bs = cst + (size_t)st * WIN_HALF;
                    const double* Ap = phi + hb * 16;
                    if (tn * MO_BN + wn0 < nsp)   // (a warp whose 16 columns lie beyond the orbitals only keeps the ring going)
#pragma unroll
                    for (int kk = 0; kk < MO_BK / 8; kk++) {
                        double af[WIN_MT], bf[2];
#pragma unroll
                        for (int mi = 0; mi < WIN_MT; mi++) {
                            const int r = mi * 8 + lr;
                            af[mi] = r < rows ? Ap[(size_t)r * L.phi_ld + kk * 4 + lc] : 0.0;
                        }
#pragma unroll
                        for (int j = 0; j < 2; j++) bf[j] = Bs[(kk * 4 + lc) * MO_BLD + wn0 + j * 8 + lr];
#pragma unroll
                        for (int mi = 0; mi < WIN_MT; mi++)
#pragma unroll
                            for (int j = 0; j < 2; j++) dmma884(acc[mi][j][0], acc[mi][j][1], af[mi], bf[j]);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[st]);
                }
#pragma unroll
                for (int mi = 0; mi < WIN_MT; mi++) {
                    const int r = mi * 8 + lr;
                    if (r < rows) {
                        const int g = r / 5, c = r - g * 5;
                        double* vrow = wd.V + ((size_t)(w0 + g) * 5 + c) * wd.ldv;
#pragma unroll
                        for (int j = 0; j < 2; j++) {
                            const int col = tn * MO_BN + wn0 + j * 8 + lc * 2;
                            if (col < nsp) *reinterpret_cast<double2*>(vrow + col) = make_double2(acc[mi][j][0], acc[mi][j][1]);
                        }
                    }
                }
            }
        }
        __syncthreads();   // V is written
    }
}

}  // namespace qmc
