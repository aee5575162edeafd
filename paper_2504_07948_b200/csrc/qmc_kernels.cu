// qmc_kernels.cu -- the CUDA kernels of the batched electron move (sm_100a) and their launchers.
// Rows a1-a9 of SURVEY.md 8(a); formulas follow BASELINE.json north_star / DESIGN.md "Readings".
#include "qmc_kernels.cuh"

#include <math.h>

#include <type_traits>

#include "gemm_f64.cuh"
#include "mo_streamk.cuh"
#include "device_utils.cuh"
#include "step_kernel.cuh"
#include "step_onepass.cuh"
#include "block_inverse.cuh"
#include "dmc_kernels.cuh"
#include "small_sweep.cuh"
#include "force_kernels.cuh"
#include "nlpp_kernels.cuh"

#ifndef QMC_UPD_BM
// flush update GEMM tile, measured on B200 at config 2 (k = 64): 64x64 CTA tile, 16x32 warp tiles, 3 stages = 2.50 ms per
// flush against 2.87 ms for 128x64 / 64x32 / 2 and 3.31 ms for 128x128 / 32x64 / 2 (small tiles, several CTAs per SM)
#define QMC_UPD_BM 64
#define QMC_UPD_BN 64
#define QMC_UPD_STAGES 3
#endif
#ifndef QMC_UPD_WM
#define QMC_UPD_WM 16
#define QMC_UPD_WN 32
#endif
#ifndef QMC_MO_CARVEOUT
#define QMC_MO_CARVEOUT 86   // percent of 228 KB: the 196 KB split
#endif
#ifndef QMC_Y_STAGES
#define QMC_Y_STAGES 3
#endif

namespace qmc {

thread_local uint64_t g_launches = 0;
#define COUNT_LAUNCH() (++g_launches)

// ------------------------------------------------------------------------------------------------
// a3: basis functions (value, gradient, laplacian) at the proposed positions          [north_star item 1]
// One CTA builds one A stage of the MO contraction -- 128 rows (row = point*5 + component) x 32 functions,
// rows padded to 36 doubles -- in shared memory and hands it to the TMA engine as ONE contiguous 36,864 B
// bulk store (cp.async.bulk.global.shared::cta, SASS UBLKCP), so HBM sees only full-line writes.  Threads
// take (point, shell) pairs of the tile; a shell that straddles two k-blocks is evaluated by both.
__device__ __forceinline__ void bulk_s2g(void* gmem_dst, const void* smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gmem_dst), "r"(smem_u32(smem_src)), "r"(bytes)
                 : "memory");
}

// Rows of a stage built by one CTA when the stage maximum is not recorded, and threads / resident CTAs per row count.
// Measured on B200 at config 2 (us per launch, live): 128 rows with 256 threads x 4 CTAs per SM 22.6, with 192 threads x 5
// CTAs per SM 21.4 (kept: one more stage draining through the TMA engine while the others compute), 64 rows with 128
// threads x 8 CTAs per SM 22.9.
#ifndef QMC_BASIS_TR
#define QMC_BASIS_TR 128
#endif
template <int TR> constexpr int BASIS_NT = TR == 128 ? 192 : 128;
template <int TR> constexpr int BASIS_MINB = TR == 128 ? 5 : 8;
constexpr int BASIS_SLD = 14;  // doubles per staged shell record (12 + 2 of padding)
// NC rows per point: 5 (value, gradient, Laplacian: the sweep) or 1 (values only: the quadrature points of row f3);
// TR rows of the stage per CTA (128: the whole stage; 64: half of it, twice as many CTAs of half the threads)
template <int NC, int TR> constexpr int BASIS_MAXPT = (TR + NC - 1) / NC + 1;  // points that can touch one TR-row piece

// exp(x) for the arguments of the primitives, x = -alpha t <= 0 (or NaN, which is returned).  The library exp spent
// half of the kernel's instructions (ncu source page: about 65 per call, a third of them moves of its constants); this
// one is 22: n = round(x log2 e) by the 1.5 * 2^52 trick, r = x - n ln 2 in two fused steps (ln 2 split hi + lo),
// the Taylor polynomial of degree 13 on |r| <= ln 2 / 2 (remainder 4e-18), 2^n added into the exponent field.  Maximum
// error measured against long-double exp on 2e7 arguments in [-708, 0]: 0.87 ulp (the library's bound is 1 ulp).
// Below -708 the result (under 3e-308, the subnormal range) is 0.
__constant__ double EXP_TAYLOR[14] = {1.0, 1.0, 1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0, 1.0 / 5040.0, 1.0 / 40320.0, 1.0 / 362880.0,
                                        1.0 / 3628800.0, 1.0 / 39916800.0, 1.0 / 479001600.0, 1.0 / 6227020800.0};  // 1 / k!
struct Exp3 {
    double a, b, c;
};
__device__ __forceinline__ Exp3 exp_neg3(double xa, double xb, double xc) {
    const double MAGIC = 6755399441055744.0, L2E = 1.4426950408889634, LN2_HI = 0.6931471805599453, LN2_LO = 2.3190468138462996e-17;
    const double ta = fma(xa, L2E, MAGIC), tb = fma(xb, L2E, MAGIC), tc = fma(xc, L2E, MAGIC);
    const double na = ta - MAGIC, nb = tb - MAGIC, nc = tc - MAGIC;
    const double ra = fma(na, -LN2_LO, fma(na, -LN2_HI, xa)), rb = fma(nb, -LN2_LO, fma(nb, -LN2_HI, xb)), rc = fma(nc, -LN2_LO, fma(nc, -LN2_HI, xc));
    const double* K = EXP_TAYLOR;  // constant-bank operands of the DFMAs
    double pa = K[13], pb = K[13], pc = K[13];
#pragma unroll
    for (int k = 12; k >= 0; k--) {  // three independent chains
        pa = fma(pa, ra, K[k]);
        pb = fma(pb, rb, K[k]);
        pc = fma(pc, rc, K[k]);
    }
    Exp3 e;
    e.a = __hiloint2double(__double2hiint(pa) + (__double2loint(ta) << 20), __double2loint(pa));
    e.b = __hiloint2double(__double2hiint(pb) + (__double2loint(tb) << 20), __double2loint(pb));
    e.c = __hiloint2double(__double2hiint(pc) + (__double2loint(tc) << 20), __double2loint(pc));
    if (!(xa >= -708.0)) e.a = xa != xa ? xa : 0.0;
    if (!(xb >= -708.0)) e.b = xb != xb ? xb : 0.0;
    if (!(xc >= -708.0)) e.c = xc != xc ? xc : 0.0;
    return e;
}

// Work items are (point, shell) pairs, ordered s-shells | p-shells | d-shells of the k-block, so a warp mixes
// shell types only at the two boundaries (no divergence in the angular code elsewhere).  The radial triple (three FP64 exp per pair -- the expensive part,
// issued as three independent chains) is computed once per shell and used from registers by its 2l+1 functions.
// The k-block's shell records (fixed 32 slots per block, so their load does not wait for the counts) are staged in
// shared memory once per CTA.
template <bool TMAX, int NC, int TR>  // TMAX: also record the largest |entry| of the stage in tilemax [MT][KB] (optional screening of the contraction)
__global__ void __launch_bounds__(BASIS_NT<TR>, BASIS_MINB<TR>) k_basis(SysDev s, const double* __restrict__ pts, int n_points, double* __restrict__ out,
                                                            double* __restrict__ tilemax) {
    static_assert(TR == MO_BM || (TR == MO_BM / 2 && !TMAX), "a CTA builds a whole stage, or half of one when no stage maximum is recorded");
    constexpr int BASIS_THREADS = BASIS_NT<TR>;
    __shared__ __align__(128) double tile[TR * MO_ALD];  // [TR][36]
    __shared__ double spt[3 * BASIS_MAXPT<NC, TR> + 3];
    __shared__ unsigned long long smax;  // bit pattern of a non-negative double: integer order = numeric order
    // rows of 14 doubles: the 16-byte reads of eight neighbouring records fall into distinct banks
    __shared__ __align__(16) double slist[32 * BASIS_SLD];
    if (threadIdx.x == 0) smax = 0ull;
    double vmax = 0.0;
    const int kb = blockIdx.x, tm = blockIdx.y, tid = threadIdx.x;
    const int4 cnt = s.kb_counts[kb];  // x, y, z = number of s, p, d shells of the block
    for (int i = tid; i < 32 * 6; i += BASIS_THREADS) {  // all 32 slots, whatever the counts: a 16-byte piece per thread
        const int sh = i / 6, j = i - sh * 6;
        reinterpret_cast<double2*>(slist + sh * BASIS_SLD)[j] = __ldg(reinterpret_cast<const double2*>(s.kb_list + kb * 32) + i);
    }
    const int row_lo = tm * TR;  // tm counts TR-row pieces
    const int pt_lo = row_lo / NC;
    int pt_hi = (row_lo + TR + NC - 1) / NC;
    if (pt_hi > n_points) pt_hi = n_points;
    const int npt = pt_hi - pt_lo;
    const int f_lo = kb * MO_BK;
    if (row_lo + TR <= NC * n_points && f_lo + MO_BK <= s.n_basis) {
        // every (row, function) of the tile gets written below: only the 4 padding columns need zeros
        for (int i = tid; i < TR * 2; i += BASIS_THREADS)
            reinterpret_cast<double2*>(tile + (i >> 1) * MO_ALD + MO_BK)[i & 1] = make_double2(0.0, 0.0);
    } else {
        for (int i = tid; i < TR * MO_ALD / 2; i += BASIS_THREADS) reinterpret_cast<double2*>(tile)[i] = make_double2(0.0, 0.0);
    }
    for (int i = tid; i < 3 * npt; i += BASIS_THREADS) spt[i] = pts[3 * pt_lo + i];
    __syncthreads();
    const int r_base = pt_lo * NC - row_lo;
    const int n0 = npt * cnt.x, n1 = n0 + npt * cnt.y, n2 = n1 + npt * cnt.z;
    const float icx = 1.0f / (float)cnt.x, icy = 1.0f / (float)cnt.y, icz = 1.0f / (float)cnt.z;  // a count of 0: never used
    for (int q = tid; q < n2; q += BASIS_THREADS) {
        int L, qq, c, base;
        float ic;
        if (q < n0) { L = 0; qq = q; c = cnt.x; ic = icx; base = 0; }
        else if (q < n1) { L = 1; qq = q - n0; c = cnt.y; ic = icy; base = cnt.x; }
        else { L = 2; qq = q - n1; c = cnt.z; ic = icz; base = cnt.x + cnt.y; }
        // qq / c without the 45-instruction integer division: c <= 32 and qq < 129 * 32, so (qq + 1/2) / c is at least
        // 1 / 64 away from an integer and the float product (error below 1e-3) truncates to the quotient
        const int pi = (int)(((float)qq + 0.5f) * ic);
        const KbShell rec = *reinterpret_cast<const KbShell*>(slist + (base + qq - pi * c) * BASIS_SLD);
        const double x = spt[3 * pi] - rec.x, y = spt[3 * pi + 1] - rec.y, z = spt[3 * pi + 2] - rec.z;
        const double t = x * x + y * y + z * z;
        // accumulation order p = 0, 1, 2, ... as in the definition of g, g', g''
        const Exp3 ex = exp_neg3(-rec.a[0] * t, -rec.a[1] * t, -rec.a[2] * t);
        const double e0 = rec.c[0] * ex.a, e1 = rec.c[1] * ex.b, e2 = rec.c[2] * ex.c;
        double g = e0, g1 = -(rec.a[0] * e0), g2 = rec.a[0] * rec.a[0] * e0;
        g += e1; g1 -= rec.a[1] * e1; g2 += rec.a[1] * rec.a[1] * e1;
        g += e2; g1 -= rec.a[2] * e2; g2 += rec.a[2] * rec.a[2] * e2;
        for (int p = 3; p < rec.nprim; p++) {
            const double al = __ldg(s.alpha + rec.poff + p);
            const double e = __ldg(s.coef + rec.poff + p) * exp(-al * t);
            g += e;
            g1 -= al * e;
            g2 += al * al * e;
        }
        const int r0 = r_base + pi * NC;  // local row of the value component (may be < 0 or > 123)
        const int c0 = rec.f0 - f_lo;
        const double lapfac = (double)(4 * L + 6) * g1 + 4.0 * t * g2;
        const double tg1 = 2.0 * g1;
        // CHK = false: shell and point lie wholly inside the stage (the usual case) -- stores at compile-time offsets
        // from one address, no range tests; CHK = true: the edges of the stage
        auto body = [&](auto CHK) {
            constexpr bool chk = decltype(CHK)::value;
            double* const t0 = tile + r0 * MO_ALD + c0;
            auto emit = [&](int m, double S, double Sx, double Sy, double Sz) {
                if (chk && (c0 + m < 0 || c0 + m >= MO_BK)) return;
                const double v[5] = {S * g, g * Sx + tg1 * S * x, g * Sy + tg1 * S * y, g * Sz + tg1 * S * z, S * lapfac};
#pragma unroll
                for (int k = 0; k < NC; k++)
                    if (!chk || (r0 + k >= 0 && r0 + k < TR)) {
                        t0[k * MO_ALD + m] = v[k];
                        if (TMAX) vmax = fmax(vmax, v[k] == v[k] ? fabs(v[k]) : INFINITY);  // a NaN stage is never screened out
                    }
            };
            const double s3 = 1.7320508075688772;
            if (L == 0) {
                emit(0, 1.0, 0.0, 0.0, 0.0);
            } else if (L == 1) {
                emit(0, x, 1.0, 0.0, 0.0);
                emit(1, y, 0.0, 1.0, 0.0);
                emit(2, z, 0.0, 0.0, 1.0);
            } else {
                emit(0, s3 * x * y, s3 * y, s3 * x, 0.0);
                emit(1, s3 * y * z, 0.0, s3 * z, s3 * y);
                emit(2, z * z - 0.5 * (x * x + y * y), -x, -y, 2.0 * z);
                emit(3, s3 * x * z, s3 * z, 0.0, s3 * x);
                emit(4, (0.5 * s3) * (x * x - y * y), s3 * x, -s3 * y, 0.0);
            }
        };
        if (r0 >= 0 && r0 + NC <= TR && c0 >= 0 && c0 + 2 * L + 1 <= MO_BK) body(std::false_type{});
        else body(std::true_type{});
    }
    if (TMAX) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) vmax = fmax(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        if ((tid & 31) == 0) atomicMax(&smax, (unsigned long long)__double_as_longlong(vmax));
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // generic-proxy smem writes -> visible to the TMA engine
    __syncthreads();
    if (tid == 0) {
        if (TMAX) tilemax[tm * s.kb + kb] = __longlong_as_double((long long)smax);  // TR = 128 here
        const int stage = row_lo / MO_BM, r_in = row_lo - stage * MO_BM;
        bulk_s2g(out + ((long)stage * s.kb + kb) * MO_A_STAGE + r_in * MO_ALD, tile, TR * MO_ALD * sizeof(double));
        asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory");  // smem must outlive the read
    }
}

// The buffer holds whole 128-row stages: with TR = 64 an odd number of pieces leaves the lower half of the last stage
// unwritten, so the grid always covers whole stages (a piece beyond the last point stores zeros).
cudaError_t launch_basis(const SysDev& s, const double* pts, int n_points, double* PhiT, double* tilemax, cudaStream_t st) {
    if (n_points == 0) return cudaSuccess;
    const int stages = (5 * n_points + MO_BM - 1) / MO_BM;
    if (tilemax) k_basis<true, 5, MO_BM><<<dim3(s.kb, stages), BASIS_NT<MO_BM>, 0, st>>>(s, pts, n_points, PhiT, tilemax);
    else k_basis<false, 5, QMC_BASIS_TR><<<dim3(s.kb, stages * (MO_BM / QMC_BASIS_TR)), BASIS_NT<QMC_BASIS_TR>, 0, st>>>(s, pts, n_points, PhiT, nullptr);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
// values only: row = point
cudaError_t launch_basis_values(const SysDev& s, const double* pts, int n_points, double* PhiT, cudaStream_t st) {
    if (n_points == 0) return cudaSuccess;
    const int stages = (n_points + MO_BM - 1) / MO_BM;
    k_basis<false, 1, QMC_BASIS_TR><<<dim3(s.kb, stages * (MO_BM / QMC_BASIS_TR)), BASIS_NT<QMC_BASIS_TR>, 0, st>>>(s, pts, n_points, PhiT, nullptr);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

}  // namespace qmc
#include "window_kernel.cuh"   // the mid-size path: needs exp_neg3 above
namespace qmc {

// one delay window of one spin in one launch (window_kernel.cuh); false: the system does not fit that path
bool window_path_ok(const SysDev& s, const WalkDev& wd, int kp) {
    const int nspm = s.nsp[0] > s.nsp[1] ? s.nsp[0] : s.nsp[1];
    if (nspm > 256) return false;
    // A CTA holds 4 walkers and an SM one CTA: beyond two waves of CTAs the per-electron kernels have rows enough to run
    // efficiently and win (measured: 152 electrons x 4320 walkers 36.5 ms per sweep per electron against 41.5 ms here;
    // configs[1], 512 walkers: 17 ms against 12.3 ms).
    int dev = 0, n_sm = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (wd.W > 2 * WIN_G * n_sm) return false;
    return window_smem_bytes(nspm, kp, s.nbp) <= 227 * 1024;
}
cudaError_t launch_window(const SysDev& s, const WalkDev& wd, int spin, int p_first, int n_steps, long log_base, int W_total, uint32_t step,
                          double tau, cudaStream_t st) {
    static SmemAttr attr;
    const size_t smem = window_smem_bytes(s.nsp[spin], wd.kp, s.nbp);
    cudaError_t e = attr.ensure(k_window, smem);
    if (e != cudaSuccess) return e;
    WinArgs a;
    a.spin = spin; a.p_first = p_first; a.n_steps = n_steps; a.log_base = log_base; a.W_total = W_total; a.step = step; a.tau = tau; a.sqrt_tau = sqrt(tau);
    k_window<<<(wd.W + WIN_G - 1) / WIN_G, WIN_THREADS, smem, st>>>(s, wd, a);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a4: MO rows V = Phi * C_s: persistent stream-K FP64 DMMA GEMM (mo_streamk.cuh)       [north_star item 2]
size_t phiT_bytes(const SysDev& s, int rows) { return (size_t)((rows + MO_BM - 1) / MO_BM) * s.kb * MO_A_STAGE * sizeof(double); }
size_t mo_ws_bytes(int grid) { return (size_t)grid * MO_WS_DOUBLES * sizeof(double); }
int mo_grid_for(const SysDev& s, int spin, int rows, int n_sm) {
    const long total = (long)((rows + MO_BM - 1) / MO_BM) * s.nt[spin] * s.kb;
    return (int)(total < n_sm ? total : n_sm);
}

// Screening plan of one contraction: a thread per row tile keeps the k-blocks whose largest entry reaches theta
// (ascending; at least one, so every output tile is written), thread 0 builds the prefix of iterations.
__global__ void __launch_bounds__(256) k_mo_plan(const double* __restrict__ tilemax, int MT, int KB, int NT, double theta, int* cnt, int* pre,
                                                 int* kbl, unsigned long long* work) {
    for (int tm = threadIdx.x; tm < MT; tm += blockDim.x) {
        int c = 0;
        for (int kb = 0; kb < KB; kb++)
            if (!(tilemax[(long)tm * KB + kb] < theta)) kbl[(long)tm * KB + c++] = kb;
        if (c == 0) { kbl[(long)tm * KB] = 0; c = 1; }
        cnt[tm] = c;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int tm = 0; tm < MT; tm++) { pre[tm] = acc; acc += NT * cnt[tm]; }
        pre[MT] = acc;
        atomicAdd(&work[0], (unsigned long long)acc);   // (the lanes of a crowd plan concurrently)
        atomicAdd(&work[1], (unsigned long long)MT * NT * KB);
    }
}

cudaError_t launch_mo_plan(const SysDev& s, int spin, const WalkDev& wd, int rows, cudaStream_t st) {
    const int MT = (rows + MO_BM - 1) / MO_BM;
    k_mo_plan<<<1, 256, 0, st>>>(wd.tilemax, MT, s.kb, s.nt[spin], wd.screen_theta, wd.plan_cnt, wd.plan_pre, wd.plan_kb, wd.mo_work);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// plan: NULL for the dense contraction, else the walker set whose plan_* buffers launch_mo_plan has just filled
cudaError_t launch_mo(const SysDev& s, int spin, const double* PhiT, int rows, double* V, long ldv, double* ws, unsigned* flags,
                      int grid, unsigned epoch, const WalkDev* plan, cudaStream_t st, unsigned long long* trace) {
    static SmemAttr attr[3];
    // shared-memory split of an SM that holds a contraction CTA: room for the other lane's step (33 KB) or basis (42 KB) CTA
    constexpr int CARVE = QMC_MO_CARVEOUT;
    cudaError_t ea = attr[0].ensure(k_mo_streamk<false, false>, MO_SMEM_BYTES, CARVE);
    if (ea == cudaSuccess) ea = attr[1].ensure(k_mo_streamk<true, false>, MO_SMEM_BYTES, CARVE);
    if (ea == cudaSuccess) ea = attr[2].ensure(k_mo_streamk<false, true>, MO_SMEM_BYTES, CARVE);
    if (ea != cudaSuccess) return ea;
    MoArgs g;
    g.PhiT = PhiT; g.CT = s.CT[spin]; g.V = V; g.ldv = ldv;
    g.M = rows; g.N = s.nsp[spin];
    g.MT = (rows + MO_BM - 1) / MO_BM; g.NT = s.nt[spin]; g.KB = s.kb;
    g.ws = ws; g.flags = flags; g.epoch = epoch; g.trace = trace;
    g.plan_cnt = plan ? plan->plan_cnt : nullptr; g.plan_pre = plan ? plan->plan_pre : nullptr; g.plan_kb = plan ? plan->plan_kb : nullptr;
    if (grid < 1) return cudaSuccess;
    // few iterations per CTA: 64-row tiles, so that a tile is split over fewer CTAs and the partial sums are smaller
    // ... or when the last 128-row tile would be at least half padding (config 3: 320 rows = five 64-row tiles, not three of 128)
    const bool half = !plan && ((long)g.MT * g.NT * g.KB < 16L * grid || g.MT * MO_BM - rows >= 64);
    if (half) g.MT = (rows + 63) / 64;
    if (plan) k_mo_streamk<true, false><<<grid, MO_THREADS, MO_SMEM_BYTES, st>>>(g);
    else if (half) k_mo_streamk<false, true><<<grid, MO_THREADS, MO_SMEM_BYTES, st>>>(g);
    else k_mo_streamk<false, false><<<grid, MO_THREADS, MO_SMEM_BYTES, st>>>(g);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a1 + a2 + a5 + a6 + a7: the fused per-walker step kernel lives in step_kernel.cuh
cudaError_t launch_step(const SysDev& s, const WalkDev& wd, int spin, int p_acc, int p_prop, long log_off, uint32_t step, double tau,
                        int commit, cudaStream_t st) {
    static SmemAttr attr[3], attr1[2];
    if (step1_fits(s.nsp[spin], wd.kp, wd.onepass != 0)) {   // large systems: the delay window read once (step_onepass.cuh)
        const int pt1 = step1_threads(s.nsp[spin], wd.kp);
        const size_t smem1 = step1_smem_bytes(s.nsp[spin], wd.kp, pt1);
        const cudaError_t e1 = pt1 == S1_PT_SMALL ? attr1[0].ensure(k_step1p<S1_PT_SMALL>, smem1) : attr1[1].ensure(k_step1p<S1_PT_LARGE>, smem1);
        if (e1 != cudaSuccess) return e1;
        if (pt1 == S1_PT_SMALL) k_step1p<S1_PT_SMALL><<<wd.W, S1_PT_SMALL, smem1, st>>>(s, wd, spin, p_acc, p_prop, log_off, step, tau, sqrt(tau), commit);
        else k_step1p<S1_PT_LARGE><<<wd.W, S1_PT_LARGE, smem1, st>>>(s, wd, spin, p_acc, p_prop, log_off, step, tau, sqrt(tau), commit);
        COUNT_LAUNCH();
        return cudaGetLastError();
    }
    const int pt = step_threads(s.nsp[spin], wd.lean != 0);
    const size_t smem = step_smem_bytes(s.nsp[spin], wd.kp, wd.lean != 0);
    const cudaError_t er = pt == 512 ? attr[2].ensure(k_step<512>, smem) : (pt == 256 ? attr[1].ensure(k_step<256>, smem) : attr[0].ensure(k_step<128>, smem));
    if (er != cudaSuccess) return er;
    if (pt == 512) k_step<512><<<wd.W, 512, smem, st>>>(s, wd, spin, p_acc, p_prop, log_off, step, tau, sqrt(tau), commit);
    else if (pt == 256) k_step<256><<<wd.W, 256, smem, st>>>(s, wd, spin, p_acc, p_prop, log_off, step, tau, sqrt(tau), commit);
    else k_step<128><<<wd.W, 128, smem, st>>>(s, wd, spin, p_acc, p_prop, log_off, step, tau, sqrt(tau), commit);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a8: delayed rank-k flush as FP64 GEMMs                                           [north_star item 5]
//   YT[q][n] = delta(q, p_n) - AinvT0[q][:] . Vbuf[n][:]           (n < m; columns n >= m are zero)
//   W2[l][j] = sum_n SinvT[l][n] Wbuf[n][j]
//   AinvT[q][j] += sum_l YT[q][l] W2[l][j]
struct EpiY {
    static constexpr bool preload = false;
    const int* plist; const int* mcount; int kp;
    __device__ bool skip(int b) const { return mcount[b] == 0; }
    __device__ void operator()(int b, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row >= M || col >= N) return;
        const int m = mcount[b];
        const int* pl = plist + (long)b * kp;
        v0 = (col < m) ? (((pl[col] == row) ? 1.0 : 0.0) - v0) : 0.0;      // stored negated: the update is A^-T += YT * W2
        v1 = (col + 1 < m) ? (((pl[col + 1] == row) ? 1.0 : 0.0) - v1) : 0.0;
        *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(v0, v1);
    }
};
struct EpiStoreSkip {
    static constexpr bool preload = false;
    const int* mcount;
    __device__ bool skip(int b) const { return mcount[b] == 0; }
    __device__ void operator()(int, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row < M && col < N) *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(v0, v1);
    }
};
struct EpiAccumSkip {  // C += A*B: accumulators preloaded from C, plain store
    static constexpr bool preload = true;
    const int* mcount;
    __device__ bool skip(int b) const { return mcount[b] == 0; }
    __device__ void operator()(int, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row < M && col < N) *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(v0, v1);
    }
};

using CfgY16 = GemmCfg<128, 16, 16, 16, true, 4>;
using CfgY32 = GemmCfg<128, 32, 16, 32, true, 4>;
using CfgY64 = GemmCfg<128, 64, 32, 32, true, QMC_Y_STAGES>;
using CfgY128 = GemmCfg<128, 128, 64, 32, true, 4>;
using CfgW2 = GemmCfg<64, 128, 32, 32, false, 3>;
using CfgUpd = GemmCfg<128, 128, 64, 32, false, 3>;   // Newton-Schulz at creation
using CfgAcc = GemmCfg<QMC_UPD_BM, QMC_UPD_BN, QMC_UPD_WM, QMC_UPD_WN, false, QMC_UPD_STAGES>;  // flush update: several CTAs per SM

__global__ void k_window_reset(WalkDev wd) {
    const int w = blockIdx.x;
    double* Si = wd.SinvT + (long)w * wd.kp * wd.kp;
    for (int i = threadIdx.x; i < wd.kp * wd.kp; i += blockDim.x) Si[i] = 0.0;
    if (threadIdx.x == 0) wd.mcount[w] = 0;
}

cudaError_t launch_window_reset(const WalkDev& wd, cudaStream_t st) {
    k_window_reset<<<wd.W, 256, 0, st>>>(wd);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// Flush of a SHORT window (at most FLUSH_SMALL_M moves pending: delay_k <= 4) in one kernel that reads A^-T once.  Row q of
// the updated inverse needs row q of the old one only -- YT[q][:] = delta - AinvT0[q][:] . Vbuf^T, then AinvT[q][:] += YT[q][:] W2
// -- and for a short window Vbuf and W2 = SinvT Wbuf (m rows each) fit in shared memory: a warp reads its row, forms the m dot
// products, reads the row again (L1) and writes it back updated.  The three GEMMs read A^-T twice and write it once, and a
// rank-1 "GEMM" is a matrix-vector product on tensor-core tiles that are fifteen-sixteenths padding; at delay_k = 1..4 the flush
// is bound by HBM, so this is the whole difference (configs[4] at 256 walkers: k = 1 148 k -> 200 k moves/s, the flush at 5.7 TB/s;
// k = 4 323 k -> 351 k).  With eight rows the shared-memory reads of the 2 m vectors per row cost more than the second read of
// A^-T (k = 8: 316 k against 398 k with the GEMMs).  Grid (row chunks, walkers).
constexpr int FLUSH_SMALL_M = 4, FLUSH_SMALL_ROWS = 64;
inline size_t flush_small_smem(int nsp, int m_cap) { return ((size_t)2 * m_cap * nsp + (size_t)m_cap * m_cap + m_cap + 2) * sizeof(double); }
__global__ void __launch_bounds__(256) k_flush_small(WalkDev wd, double* __restrict__ Ainv, int nsp, int m_cap) {
    extern __shared__ __align__(16) double fsm[];
    const int w = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int m = wd.mcount[w], kp = wd.kp, n2 = nsp >> 1;
    if (m == 0) return;
    if (m > m_cap || m > FLUSH_SMALL_M) {   // (never: the scheduler passes delay_k; raise the walker's sticky flag rather than overrun shared memory)
        if (tid == 0) wd.flags[w] = 1u;
        return;
    }
    double* Vs = fsm;
    double* W2s = Vs + (size_t)m_cap * nsp;
    double* Ss = W2s + (size_t)m_cap * nsp;
    int* pl = reinterpret_cast<int*>(Ss + m_cap * m_cap);
    const double* Vb = wd.Vbuf + (long)w * kp * nsp;
    const double* Wb = wd.Wbuf + (long)w * kp * nsp;
    for (int i = tid; i < m * n2; i += 256) reinterpret_cast<double2*>(Vs)[i] = __ldg(reinterpret_cast<const double2*>(Vb) + i);   // rows 0 .. m-1 are contiguous
    for (int i = tid; i < m * m; i += 256) Ss[i] = wd.SinvT[(long)w * kp * kp + (i / m) * kp + (i % m)];
    if (tid < m) pl[tid] = wd.plist[(long)w * kp + tid];
    __syncthreads();
    for (int j2 = tid; j2 < n2; j2 += 256) {   // W2[l][j] = sum_n SinvT[l][n] Wbuf[n][j]
        double2 wv[FLUSH_SMALL_M];
#pragma unroll
        for (int n = 0; n < FLUSH_SMALL_M; n++) wv[n] = n < m ? __ldg(reinterpret_cast<const double2*>(Wb + (long)n * nsp) + j2) : make_double2(0.0, 0.0);
#pragma unroll
        for (int l = 0; l < FLUSH_SMALL_M; l++) {
            if (l >= m) break;
            double2 acc = make_double2(0.0, 0.0);
#pragma unroll
            for (int n = 0; n < FLUSH_SMALL_M; n++)
                if (n < m) { const double c = Ss[l * m + n]; acc.x += c * wv[n].x; acc.y += c * wv[n].y; }
            reinterpret_cast<double2*>(W2s + (size_t)l * nsp)[j2] = acc;
        }
    }
    __syncthreads();
    const int q0 = blockIdx.x * FLUSH_SMALL_ROWS;
    const int q1 = q0 + FLUSH_SMALL_ROWS < nsp ? q0 + FLUSH_SMALL_ROWS : nsp;
    for (int q = q0 + warp; q < q1; q += 8) {
        double2* row = reinterpret_cast<double2*>(Ainv + ((long)w * nsp + q) * nsp);
        double y[FLUSH_SMALL_M];
#pragma unroll
        for (int n = 0; n < FLUSH_SMALL_M; n++) y[n] = 0.0;
        for (int j2 = lane; j2 < n2; j2 += 32) {
            const double2 a = row[j2];
#pragma unroll
            for (int n = 0; n < FLUSH_SMALL_M; n++)
                if (n < m) { const double2 v = reinterpret_cast<const double2*>(Vs + (size_t)n * nsp)[j2]; y[n] += a.x * v.x + a.y * v.y; }
        }
#pragma unroll
        for (int n = 0; n < FLUSH_SMALL_M; n++)
            if (n < m) y[n] = (pl[n] == q ? 1.0 : 0.0) - warp_sum(y[n]);
        for (int j2 = lane; j2 < n2; j2 += 32) {
            double2 a = row[j2];   // (L1: this warp has just read the row)
#pragma unroll
            for (int l = 0; l < FLUSH_SMALL_M; l++)
                if (l < m) { const double2 u = reinterpret_cast<const double2*>(W2s + (size_t)l * nsp)[j2]; a.x += y[l] * u.x; a.y += y[l] * u.y; }
            row[j2] = a;
        }
    }
}

cudaError_t launch_flush(const SysDev& s, const WalkDev& wd, int spin, cudaStream_t st, int max_m) {
    const int nsp = s.nsp[spin], kp = wd.kp;
    cudaError_t e;
    if (max_m >= 1 && max_m <= FLUSH_SMALL_M && flush_small_smem(nsp, max_m) <= 200 * 1024) {
        static SmemAttr attr;
        const size_t smem = flush_small_smem(nsp, max_m);
        e = attr.ensure(k_flush_small, smem);
        if (e != cudaSuccess) return e;
        k_flush_small<<<dim3((nsp + FLUSH_SMALL_ROWS - 1) / FLUSH_SMALL_ROWS, wd.W), 256, smem, st>>>(wd, wd.AinvT[spin], nsp, max_m);
        COUNT_LAUNCH();
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        return launch_window_reset(wd, st);
    }
    GemmArgs g;
    // YT = AinvT0 * Vbuf^T
    g.A = wd.AinvT[spin]; g.lda = nsp; g.strideA = (long)nsp * nsp;
    g.B = wd.Vbuf; g.ldb = nsp; g.strideB = (long)kp * nsp;
    g.C = wd.YT; g.ldc = kp; g.strideC = (long)nsp * kp;
    g.M = nsp; g.N = kp; g.K = nsp;
    EpiY ey{wd.plist, wd.mcount, kp};
    if (kp <= 16) e = gemm_f64_launch<CfgY16>(g, wd.W, ey, st);
    else if (kp <= 32) e = gemm_f64_launch<CfgY32>(g, wd.W, ey, st);
    else if (kp <= 64) e = gemm_f64_launch<CfgY64>(g, wd.W, ey, st);
    else e = gemm_f64_launch<CfgY128>(g, wd.W, ey, st);
    COUNT_LAUNCH();
    if (e != cudaSuccess) return e;
    // W2 = SinvT * Wbuf
    g.A = wd.SinvT; g.lda = kp; g.strideA = (long)kp * kp;
    g.B = wd.Wbuf; g.ldb = nsp; g.strideB = (long)kp * nsp;
    g.C = wd.W2; g.ldc = nsp; g.strideC = (long)kp * nsp;
    g.M = kp; g.N = nsp; g.K = kp;
    e = gemm_f64_launch<CfgW2>(g, wd.W, EpiStoreSkip{wd.mcount}, st);
    COUNT_LAUNCH();
    if (e != cudaSuccess) return e;
    // AinvT += YT * W2
    g.A = wd.YT; g.lda = kp; g.strideA = (long)nsp * kp;
    g.B = wd.W2; g.ldb = nsp; g.strideB = (long)kp * nsp;
    g.C = wd.AinvT[spin]; g.ldc = nsp; g.strideC = (long)nsp * nsp;
    g.M = nsp; g.N = nsp; g.K = kp;
    e = gemm_f64_launch<CfgAcc>(g, wd.W, EpiAccumSkip{wd.mcount}, st);
    COUNT_LAUNCH();
    if (e != cudaSuccess) return e;
    return launch_window_reset(wd, st);
}

// ------------------------------------------------------------------------------------------------
// a9: local energy E_L = K + V                                                     [north_star item 6]
// One warp per electron: 4 dots over the row caches, Jastrow gradient/laplacian and Coulomb sums over
// partners with warp-shuffle reductions; then a fixed-order per-walker reduction.
__global__ void __launch_bounds__(256, 4) k_eloc_elec(SysDev s, WalkDev wd) {
    const int w = blockIdx.y;
    const int e = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (e >= s.ne) return;
    const int spin = e < s.ns[0] ? 0 : 1, p = spin ? e - s.ns[0] : e;
    const int nsp = s.nsp[spin], nep = wd.nep;
    const double* arow = wd.AinvT[spin] + ((long)w * nsp + p) * nsp;
    const double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    double gx = 0, gy = 0, gz = 0, lp = 0;
    {   // 4 dot products over the row caches: 16-byte loads, 10 in flight per lane
        const double2* a2 = reinterpret_cast<const double2*>(arow);
        const double2* o1 = reinterpret_cast<const double2*>(orb + nsp);
        const double2* o2 = reinterpret_cast<const double2*>(orb + 2 * nsp);
        const double2* o3 = reinterpret_cast<const double2*>(orb + 3 * nsp);
        const double2* o4 = reinterpret_cast<const double2*>(orb + 4 * nsp);
        const int n2 = nsp >> 1;
        int j = lane;
        for (; j + 32 < n2; j += 64) {
            const double2 a = __ldg(a2 + j), b = __ldg(a2 + j + 32);
            const double2 p1 = __ldg(o1 + j), q1 = __ldg(o1 + j + 32), p2 = __ldg(o2 + j), q2 = __ldg(o2 + j + 32);
            const double2 p3 = __ldg(o3 + j), q3 = __ldg(o3 + j + 32), p4 = __ldg(o4 + j), q4 = __ldg(o4 + j + 32);
            gx += p1.x * a.x + p1.y * a.y + q1.x * b.x + q1.y * b.y;
            gy += p2.x * a.x + p2.y * a.y + q2.x * b.x + q2.y * b.y;
            gz += p3.x * a.x + p3.y * a.y + q3.x * b.x + q3.y * b.y;
            lp += p4.x * a.x + p4.y * a.y + q4.x * b.x + q4.y * b.y;
        }
        for (; j < n2; j += 32) {
            const double2 a = __ldg(a2 + j), p1 = __ldg(o1 + j), p2 = __ldg(o2 + j), p3 = __ldg(o3 + j), p4 = __ldg(o4 + j);
            gx += p1.x * a.x + p1.y * a.y;
            gy += p2.x * a.x + p2.y * a.y;
            gz += p3.x * a.x + p3.y * a.y;
            lp += p4.x * a.x + p4.y * a.y;
        }
    }
    const double* Rw = wd.R + (long)w * 3 * nep;
    const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
    double jx = 0, jy = 0, jz = 0, jl = 0, pot = 0;
    const int npart = s.ne + s.n_atoms;
    // u' = a / q^2, u'' = -2ab / q^3 with q = 1 + b r: one sqrt and two divisions (1/r, 1/q) per pair
    for (int k = lane; k < npart; k += 32) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double ir = 1.0 / r, iq = 1.0 / (1.0 + P.b * r);
            const double du = P.a * iq * iq;
            const double wgt = du * ir;
            jx += wgt * dx; jy += wgt * dy; jz += wgt * dz;
            jl += 2.0 * wgt - 2.0 * P.b * du * iq;
            if (k >= s.ne) pot += P.a * ir;         // P.a = -Z_I
            else if (k > e) pot += ir;              // each pair once
        }
    }
    gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz); lp = warp_sum(lp);
    jx = warp_sum(jx); jy = warp_sum(jy); jz = warp_sum(jz); jl = warp_sum(jl); pot = warp_sum(pot);
    if (lane == 0) {
        const double g2 = gx * gx + gy * gy + gz * gz;
        const double tx = gx + jx, ty = gy + jy, tz = gz + jz;
        const double kin = lp - g2 + jl + (tx * tx + ty * ty + tz * tz);
        wd.ebuf[((long)w * s.ne + e) * 2] = kin;
        wd.ebuf[((long)w * s.ne + e) * 2 + 1] = pot;
    }
}

__global__ void __launch_bounds__(256) k_eloc_reduce(SysDev s, WalkDev wd) {
    __shared__ double red[2 * 8];
    const int w = blockIdx.x;
    double a2[2] = {0, 0};
    for (int e = threadIdx.x; e < s.ne; e += 256) {
        a2[0] += wd.ebuf[((long)w * s.ne + e) * 2];
        a2[1] += wd.ebuf[((long)w * s.ne + e) * 2 + 1];
    }
    block_sum<256, 2>(a2, red);
    if (threadIdx.x == 0) {
        const double K = -0.5 * a2[0];
        wd.ekin[w] = K;
        wd.eloc[w] = K + (a2[1] + s.e_nn);
    }
}

cudaError_t launch_eloc(const SysDev& s, const WalkDev& wd, cudaStream_t st) {
    dim3 grid((s.ne + 7) / 8, wd.W);
    k_eloc_elec<<<grid, 256, 0, st>>>(s, wd);
    COUNT_LAUNCH();
    k_eloc_reduce<<<wd.W, 256, 0, st>>>(s, wd);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// walker creation helpers
__global__ void k_gather_rp(WalkDev wd, int e) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= wd.W) return;
    const double* Rw = wd.R + (long)w * 3 * wd.nep;
    wd.rp[3 * w] = Rw[e]; wd.rp[3 * w + 1] = Rw[wd.nep + e]; wd.rp[3 * w + 2] = Rw[2 * wd.nep + e];
}
cudaError_t launch_gather_rp(const WalkDev& wd, int e, cudaStream_t st) {
    k_gather_rp<<<(wd.W + 127) / 128, 128, 0, st>>>(wd, e);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// Orb[w][p][0..4][:] <- V[w][0..4][:], and the transposed Slater matrix T[j][p] = A[p][j] into AinvT
__global__ void k_store_init_rows(SysDev s, WalkDev wd, int spin, int p) {
    const int w = blockIdx.x, nsp = s.nsp[spin];
    const double* v = wd.V + (long)w * 5 * wd.ldv;
    double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    double* T = wd.AinvT[spin] + (long)w * nsp * nsp;
    for (int j = threadIdx.x; j < nsp; j += blockDim.x) {
        for (int c = 0; c < 5; c++) orb[c * nsp + j] = v[c * wd.ldv + j];
        if (j < s.ns[spin]) T[(long)j * nsp + p] = v[j];
    }
}
cudaError_t launch_store_init_rows(const SysDev& s, const WalkDev& wd, int spin, int p, cudaStream_t st) {
    k_store_init_rows<<<wd.W, 256, 0, st>>>(s, wd, spin, p);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// In-place Gauss-Jordan inverse with partial (row) pivoting of the n x n leading block of each matrix;
// one CTA per matrix.  logdet/sign accumulate over calls (one call per spin).
template <int NT>
__global__ void __launch_bounds__(NT) k_gj_inverse(double* Mall, long stride, int n, int ld, double* logdet, int* sign, int* status) {
    extern __shared__ double gsm[];
    double* rowk = gsm;               // [n]
    double* colk = rowk + n;          // [n]
    double* redv = colk + n;          // [NT/32]
    int* redi = (int*)(redv + NT / 32);  // [NT/32]
    int* perm = redi + NT / 32;       // [n]
    __shared__ int s_piv;
    __shared__ double s_pivval;
    double* M = Mall + (long)blockIdx.x * stride;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double lad = 0.0;
    int sg = 1;
    for (int k = 0; k < n; k++) {
        // pivot search: max |M[i][k]|, i >= k, lowest index on ties
        double best = -1.0;
        int bi = k;
        for (int i = k + tid; i < n; i += NT) {
            const double v = fabs(M[(long)i * ld + k]);
            if (v > best) { best = v; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if (lane == 0) { redv[warp] = best; redi[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            double b = redv[0];
            int r = redi[0];
            for (int q = 1; q < NT / 32; q++)
                if (redv[q] > b || (redv[q] == b && redi[q] < r)) { b = redv[q]; r = redi[q]; }
            s_piv = r;
            s_pivval = b;
            perm[k] = r;
        }
        __syncthreads();
        const int r = s_piv;
        if (!(s_pivval > 0.0)) {  // singular (or NaN)
            if (tid == 0) status[0] = -3;
            return;
        }
        // swap rows k and r; build the scaled pivot row in shared memory
        const double piv = M[(long)r * ld + k];
        __syncthreads();  // everyone has read piv before row r is overwritten
        const double pinv = 1.0 / piv;
        for (int j = tid; j < n; j += NT) {
            const double a = M[(long)r * ld + j];
            if (r != k) M[(long)r * ld + j] = M[(long)k * ld + j];
            const double v = (j == k ? 1.0 : a) * pinv;
            rowk[j] = v;
            M[(long)k * ld + j] = v;
        }
        __syncthreads();
        for (int i = tid; i < n; i += NT) {
            double f = 0.0;
            if (i != k) { f = M[(long)i * ld + k]; M[(long)i * ld + k] = 0.0; }
            colk[i] = f;
        }
        __syncthreads();
        if (tid == 0) {
            lad += log(fabs(piv));
            if (piv < 0.0) sg = -sg;
            if (r != k) sg = -sg;
        }
        // eliminate: M[i][j] -= colk[i] * rowk[j], all i != k
        for (int j = tid; j < n; j += NT) {
            const double rk = rowk[j];
#pragma unroll 4
            for (int i = 0; i < n; i++) {
                const double f = colk[i];
                if (f != 0.0) M[(long)i * ld + j] -= f * rk;
            }
        }
        __syncthreads();
    }
    // undo the row permutation as column swaps, in reverse order
    for (int k = n - 1; k >= 0; k--) {
        const int r = perm[k];
        if (r != k) {
            for (int i = tid; i < n; i += NT) {
                const double a = M[(long)i * ld + k];
                M[(long)i * ld + k] = M[(long)i * ld + r];
                M[(long)i * ld + r] = a;
            }
        }
        __syncthreads();
    }
    if (tid == 0) {
        logdet[blockIdx.x] += lad;
        sign[blockIdx.x] *= sg;
    }
}

using CfgGjb = GemmCfg<64, 64, 16, 32, false, 2>;

// Blocked inversion (block_inverse.cuh) for n >= 256 when a panel fits in shared memory; tmp: scratch of batch * stride doubles.
static cudaError_t launch_block_inverse(double* Mall, long stride, int n, int ld, int batch, double* logdet, int* sign, int* status,
                                        double* tmp, cudaStream_t st) {
    const int nb = gjb_panel_width(n);
    GjbArgs g;
    g.M = Mall; g.stride = stride; g.n = n; g.ld = ld; g.logdet = logdet; g.sign = sign; g.status = status;
    char* buf = nullptr;
    const size_t bFn = (size_t)batch * ld * GJB_NB * 8, bT = bFn, bP = (size_t)batch * GJB_NB * GJB_NB * 8, bR = (size_t)batch * ld * 4,
                 bU = (size_t)batch * ld;
    cudaError_t e = cudaMalloc((void**)&buf, bFn + bT + bP + bR + bU + 256);
    if (e != cudaSuccess) return e;
    g.Fn = (double*)buf; g.T = (double*)(buf + bFn); g.Pinv = (double*)(buf + bFn + bT);
    g.rowof = (int*)(buf + bFn + bT + bP); g.used = (unsigned char*)(buf + bFn + bT + bP + bR);
    e = cudaMemsetAsync(buf, 0, bFn + bT + bP + bR + bU, st);
    const size_t smem = gjb_panel_smem(n, nb);
    static SmemAttr panel_attr;
    if (e == cudaSuccess) e = panel_attr.ensure(k_gjb_panel, smem);
    GemmArgs ga;
    ga.A = g.Fn; ga.lda = GJB_NB; ga.strideA = (long)ld * GJB_NB;
    ga.B = g.T; ga.ldb = ld; ga.strideB = (long)GJB_NB * ld;
    ga.C = Mall; ga.ldc = ld; ga.strideC = stride;
    ga.M = ld; ga.N = ld; ga.K = GJB_NB;
    for (int k0 = 0; k0 < n && e == cudaSuccess; k0 += nb) {
        const int nbk = n - k0 < nb ? n - k0 : nb;
        k_gjb_panel<<<batch, GJB_THREADS, smem, st>>>(g, k0, nbk, nb);
        k_gjb_rows<<<dim3((ld + 255) / 256, batch), 256, 0, st>>>(g, k0, nbk);
        e = gemm_f64_launch<CfgGjb>(ga, batch, EpiAccum{}, st);
        g_launches += 3;
    }
    if (e == cudaSuccess) {
        k_gjb_permute<<<dim3((n + 255) / 256, n, batch), 256, 0, st>>>(g, tmp);
        k_gjb_copy_back<<<dim3((n + 255) / 256, n, batch), 256, 0, st>>>(g, tmp);
        k_gjb_perm_sign<<<(batch + 63) / 64, 64, 0, st>>>(g, batch);
        g_launches += 3;
        e = cudaGetLastError();
    }
    cudaError_t e2 = cudaStreamSynchronize(st);
    cudaFree(buf);
    return e != cudaSuccess ? e : e2;
}

cudaError_t launch_gj_inverse(double* Mall, long stride, int n, int ld, int batch, double* logdet, int* sign, int* status, double* tmp,
                              cudaStream_t st) {
    if (n == 0 || batch == 0) return cudaSuccess;
    if (n >= 256 && tmp && gjb_panel_width(n) >= 4) return launch_block_inverse(Mall, stride, n, ld, batch, logdet, sign, status, tmp, st);
    COUNT_LAUNCH();
    if (n >= 512) {
        constexpr int NT = 1024;
        size_t smem = (size_t)(2 * n + NT / 32) * sizeof(double) + (size_t)(NT / 32 + n) * sizeof(int);
        static SmemAttr attr;
        const cudaError_t ea = attr.ensure(k_gj_inverse<NT>, smem);
        if (ea != cudaSuccess) return ea;
        k_gj_inverse<NT><<<batch, NT, smem, st>>>(Mall, stride, n, ld, logdet, sign, status);
    } else {
        constexpr int NT = 256;
        size_t smem = (size_t)(2 * n + NT / 32) * sizeof(double) + (size_t)(NT / 32 + n) * sizeof(int);
        k_gj_inverse<NT><<<batch, NT, smem, st>>>(Mall, stride, n, ld, logdet, sign, status);
    }
    return cudaGetLastError();
}

// One Newton-Schulz step on the freshly inverted matrices: Y <- Y + (I - Y A^T) Y with Y = AinvT (= (A^T)^-1) and
// A read from the value rows of the row cache.  Two batched DMMA GEMMs; brings the Gauss-Jordan result to the
// accuracy of a backward-stable inverse (residual-limited) at ~4 N^3 flop per matrix.
struct EpiEyeMinus {
    static constexpr bool preload = false;
    int ns;
    __device__ bool skip(int) const { return false; }
    __device__ void operator()(int, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row >= M || col >= N) return;
        const double d0 = (row == col && row < ns) ? 1.0 : 0.0, d1 = (row == col + 1 && row < ns) ? 1.0 : 0.0;
        *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(d0 - v0, d1 - v1);
    }
};
struct EpiAddSrc {
    static constexpr bool preload = false;
    const double* src; long stride;
    __device__ bool skip(int) const { return false; }
    __device__ void operator()(int b, double* Cb, long ldc, int M, int N, int row, int col, double v0, double v1) const {
        if (row >= M || col >= N) return;
        const double2 y = *reinterpret_cast<const double2*>(src + (long)b * stride + (long)row * ldc + col);
        *reinterpret_cast<double2*>(Cb + (long)row * ldc + col) = make_double2(y.x + v0, y.y + v1);
    }
};
cudaError_t launch_refine_inverse(const SysDev& s, const WalkDev& wd, int spin, double* E, double* Z, cudaStream_t st) {
    const int nsp = s.nsp[spin];
    if (s.ns[spin] == 0) return cudaSuccess;
    const long mat = (long)nsp * nsp;
    GemmArgs g;
    g.A = wd.AinvT[spin]; g.lda = nsp; g.strideA = mat;
    g.B = wd.Orb[spin]; g.ldb = 5L * nsp; g.strideB = 5L * mat;   // A[p'][j] = value row of electron p'
    g.C = E; g.ldc = nsp; g.strideC = mat;
    g.M = nsp; g.N = nsp; g.K = nsp;
    cudaError_t e = gemm_f64_launch<CfgY128>(g, wd.W, EpiEyeMinus{s.ns[spin]}, st);
    COUNT_LAUNCH();
    if (e != cudaSuccess) return e;
    g.A = E; g.lda = nsp; g.strideA = mat;
    g.B = wd.AinvT[spin]; g.ldb = nsp; g.strideB = mat;
    g.C = Z; g.ldc = nsp; g.strideC = mat;
    e = gemm_f64_launch<CfgUpd>(g, wd.W, EpiAddSrc{wd.AinvT[spin], mat}, st);
    COUNT_LAUNCH();
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(wd.AinvT[spin], Z, (size_t)wd.W * mat * sizeof(double), cudaMemcpyDeviceToDevice, st);
}

// J(R) by direct sums (walker creation): one CTA per walker
__global__ void __launch_bounds__(256) k_jastrow_total(SysDev s, WalkDev wd) {
    __shared__ double red[8];
    const int w = blockIdx.x, nep = wd.nep;
    const double* Rw = wd.R + (long)w * 3 * nep;
    const int npart = s.ne + s.n_atoms;
    double a1[1] = {0.0};
    for (long idx = threadIdx.x; idx < (long)s.ne * npart; idx += 256) {
        const int i = (int)(idx / npart), k = (int)(idx % npart);
        if (k < s.ne && k <= i) continue;
        Partner P = partner(s, Rw, nep, i, k);
        const double dx = Rw[i] - P.x, dy = Rw[nep + i] - P.y, dz = Rw[2 * nep + i] - P.z;
        a1[0] += pade_u(P.a, P.b, sqrt(dx * dx + dy * dy + dz * dz));
    }
    block_sum<256, 1>(a1, red);
    if (threadIdx.x == 0) wd.logpsi[w] += a1[0];
}
cudaError_t launch_jastrow_total(const SysDev& s, const WalkDev& wd, cudaStream_t st) {
    k_jastrow_total<<<wd.W, 256, 0, st>>>(s, wd);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// nuclear repulsion sum_{I<J} Z_I Z_J / R_IJ (system constant), one CTA
__global__ void __launch_bounds__(256) k_enn(SysDev s, double* out) {
    __shared__ double red[8];
    double a1[1] = {0.0};
    const long n = (long)s.n_atoms * s.n_atoms;
    for (long idx = threadIdx.x; idx < n; idx += 256) {
        const int I = (int)(idx / s.n_atoms), J = (int)(idx % s.n_atoms);
        if (J <= I) continue;
        const double dx = s.atom_xyz[3 * I] - s.atom_xyz[3 * J], dy = s.atom_xyz[3 * I + 1] - s.atom_xyz[3 * J + 1],
                     dz = s.atom_xyz[3 * I + 2] - s.atom_xyz[3 * J + 2];
        a1[0] += s.atom_Z[I] * s.atom_Z[J] / sqrt(dx * dx + dy * dy + dz * dz);
    }
    block_sum<256, 1>(a1, red);
    if (threadIdx.x == 0) out[0] = a1[0];
}
cudaError_t launch_enn(const SysDev& s, double* out, cudaStream_t st) {
    k_enn<<<1, 256, 0, st>>>(s, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// layout conversion for the ABI
__global__ void k_import_positions(WalkDev wd, const double* __restrict__ in /* [W][ne][3] */) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)wd.W * wd.ne) return;
    const int w = (int)(idx / wd.ne), e = (int)(idx % wd.ne);
    double* Rw = wd.R + (long)w * 3 * wd.nep;
    Rw[e] = in[idx * 3]; Rw[wd.nep + e] = in[idx * 3 + 1]; Rw[2 * wd.nep + e] = in[idx * 3 + 2];
}
__global__ void k_export_positions(WalkDev wd, double* __restrict__ out) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)wd.W * wd.ne) return;
    const int w = (int)(idx / wd.ne), e = (int)(idx % wd.ne);
    const double* Rw = wd.R + (long)w * 3 * wd.nep;
    out[idx * 3] = Rw[e]; out[idx * 3 + 1] = Rw[wd.nep + e]; out[idx * 3 + 2] = Rw[2 * wd.nep + e];
}
cudaError_t launch_import_positions(const WalkDev& wd, const double* in, cudaStream_t st) {
    long n = (long)wd.W * wd.ne;
    k_import_positions<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(wd, in);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
cudaError_t launch_export_positions(const WalkDev& wd, double* out, cudaStream_t st) {
    long n = (long)wd.W * wd.ne;
    k_export_positions<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(wd, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_export_ainv(const double* __restrict__ AinvT, int W, int ns, int nsp, double* __restrict__ out) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long tot = (long)W * ns * ns;
    if (idx >= tot) return;
    const int j = (int)(idx % ns);
    const long t = idx / ns;
    const int p = (int)(t % ns), w = (int)(t / ns);
    out[idx] = AinvT[((long)w * nsp + p) * nsp + j];
}
cudaError_t launch_export_ainv(const double* AinvT, int W, int ns, int nsp, double* out, cudaStream_t st) {
    long n = (long)W * ns * ns;
    if (n == 0) return cudaSuccess;
    k_export_ainv<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(AinvT, W, ns, nsp, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_export_rows(const double* __restrict__ src, long n_rows, int width, long ld, double* __restrict__ out) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_rows * width) return;
    out[idx] = src[(idx / width) * ld + idx % width];
}
cudaError_t launch_export_rows(const double* src, long n_rows, int width, long ld, double* out, cudaStream_t st) {
    long n = n_rows * width;
    if (n == 0) return cudaSuccess;
    k_export_rows<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, n_rows, width, ld, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_tile_C(const double* __restrict__ in, int nb, int ns, double* __restrict__ CT, int kb, const int* __restrict__ fmap) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)nb * ns) return;
    const int l = (int)(idx / ns), j = (int)(idx % ns);
    CT[cT_index(fmap[l], j, kb)] = in[idx];
}
cudaError_t launch_tile_C(const double* in, int nb, int ns, double* CT, int kb, const int* fmap, cudaStream_t st) {
    long n = (long)nb * ns;
    if (n == 0) return cudaSuccess;
    k_tile_C<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, nb, ns, CT, kb, fmap);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_export_phi(const double* __restrict__ PhiT, long n_rows, int width, int kb, const int* __restrict__ fmap,
                             double* __restrict__ out) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_rows * width) return;
    out[idx] = PhiT[phiT_index(idx / width, fmap[(int)(idx % width)], kb)];
}
cudaError_t launch_export_phi(const double* PhiT, long n_rows, int width, int kb, const int* fmap, double* out, cudaStream_t st) {
    long n = n_rows * width;
    if (n == 0) return cudaSuccess;
    k_export_phi<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(PhiT, n_rows, width, kb, fmap, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_sign_to_i8(const int* __restrict__ in, int n, int8_t* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (int8_t)in[i];
}
cudaError_t launch_sign_to_i8(const int* in, int n, int8_t* out, cudaStream_t st) {
    k_sign_to_i8<<<(n + 255) / 256, 256, 0, st>>>(in, n, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_fill_int(int* p, int n, int v) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}
cudaError_t launch_fill_int(int* p, int n, int v, cudaStream_t st) {
    k_fill_int<<<(n + 255) / 256, 256, 0, st>>>(p, n, v);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// FP64 ceiling: register-resident DMMA issue loop
__global__ void k_dmma_peak(double* out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) dmma884(c[i][0], c[i][1], a, b);
    }
    double sacc = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) sacc += c[i][0] + c[i][1];
    out[(long)blockIdx.x * blockDim.x + threadIdx.x] = sacc;
}
cudaError_t launch_dmma_peak(double* out, int grid, int threads, int iters, cudaStream_t st) {
    k_dmma_peak<<<grid, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// row f1: DMC generation bookkeeping and reconfiguration (dmc_kernels.cuh)
__global__ void k_fill_double(double* p, int n, double v) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}
cudaError_t launch_fill_double(double* p, int n, double v, cudaStream_t st) {
    k_fill_double<<<(n + 255) / 256, 256, 0, st>>>(p, n, v);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
cudaError_t launch_dmc_begin(const WalkDev& wd, cudaStream_t st) {
    k_dmc_begin<<<(wd.W + 255) / 256, 256, 0, st>>>(wd);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
cudaError_t launch_dmc_weight(const WalkDev& wd, double tau, double e_trial, const double* e_trial_dev, cudaStream_t st) {
    k_dmc_weight<<<(wd.W + 255) / 256, 256, 0, st>>>(wd, tau, e_trial, e_trial_dev);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
cudaError_t launch_branch(const SysDev& s, const WalkDev& wd, int* ibuf /* [4 W + 1] */, double* e_mixed, uint32_t step, double* e_trial_dev,
                          double feedback, double* branch_log, cudaStream_t st) {
    CombOut o;
    o.source = ibuf; o.pair_dst = ibuf + wd.W; o.pair_src = ibuf + 2 * wd.W; o.mult = ibuf + 3 * wd.W; o.n_pairs = ibuf + 4 * wd.W;
    o.e_mixed = e_mixed;
    o.e_trial_dev = e_trial_dev; o.feedback = feedback; o.branch_log = branch_log;
    const size_t smem = (size_t)wd.W * 8 <= 40 * 1024 ? (size_t)wd.W * 8 : 0;
    k_comb<<<1, 256, smem, st>>>(wd, o, step);
    COUNT_LAUNCH();
    CopyArgs a;
    a.n_seg = 0;
    a.seg[a.n_seg++] = CopySeg{wd.R, 3L * wd.nep};
    for (int sp = 0; sp < 2; sp++) {
        if (s.ns[sp] == 0) continue;
        a.seg[a.n_seg++] = CopySeg{wd.AinvT[sp], (long)s.nsp[sp] * s.nsp[sp]};
        a.seg[a.n_seg++] = CopySeg{wd.Orb[sp], 5L * s.nsp[sp] * s.nsp[sp]};
    }
    const long biggest = 5L * wd.ldv * wd.ldv / 2;
    int chunks = (int)((biggest + 256L * 16 - 1) / (256L * 16));
    if (chunks < 1) chunks = 1;
    if (chunks > 512) chunks = 512;
    k_copy_walkers<<<dim3(chunks, wd.W), 256, 0, st>>>(wd, a, o);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// row f4: whole call in one launch for small systems (small_sweep.cuh).  Returns false if the system does not qualify.
bool small_path_ok(const SysDev& s, const WalkDev& wd) {
    const int nsm = s.ns[0] > s.ns[1] ? s.ns[0] : s.ns[1];
    if (nsm > 32 || s.n_basis > 512) return false;
    const size_t per_block = small_block_doubles(s, nsm) * 8, per_walker = small_walker_doubles(s, wd.nep, nsm) * 8;
    return per_block + per_walker <= 200 * 1024;
}
cudaError_t launch_sweep_small(const SysDev& s, const WalkDev& wd, int nsteps, uint32_t step0, double tau, int dmc, double e_trial,
                               const double* e_trial_dev, cudaStream_t st) {
    SmallArgs a;
    a.nsteps = nsteps; a.step0 = step0; a.tau = tau; a.sqrt_tau = sqrt(tau); a.dmc = dmc; a.e_trial = e_trial; a.e_trial_dev = e_trial_dev;
    a.nsm = s.ns[0] > s.ns[1] ? s.ns[0] : s.ns[1];
    const size_t per_block = small_block_doubles(s, a.nsm) * 8, per_walker = small_walker_doubles(s, wd.nep, a.nsm) * 8;
    // warps per block: as many as fit in ~100 KB (two blocks per SM), at most 8, and no more than needed to give every SM a block
    int wpb = (int)((100 * 1024 - per_block) / per_walker);
    if (wpb < 1) wpb = 1;
    if (wpb > 8) wpb = 8;
    while (wpb > 1 && (wd.W + wpb - 1) / wpb < 148) wpb--;
    a.wpb = wpb;
    const size_t smem = per_block + (size_t)wpb * per_walker;
    static SmemAttr attr;
    const cudaError_t ea = attr.ensure(k_sweep_small, smem);
    if (ea != cudaSuccess) return ea;
    k_sweep_small<<<(wd.W + wpb - 1) / wpb, wpb * 32, smem, st>>>(s, wd, a);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// row f2, first half (force_kernels.cuh)
cudaError_t launch_plain_C(const double* in, int nb, int ns, double* Cp, int nsp, const int* fmap, cudaStream_t st) {
    long n = (long)nb * ns;
    if (n == 0) return cudaSuccess;
    k_plain_C<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, nb, ns, Cp, nsp, fmap);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
cudaError_t launch_dlogpsi_dR(const SysDev& s, const WalkDev& wd, int spin, double* Mt, double* acc, cudaStream_t st) {
    if (s.ns[spin] > 0) {
        // Mt[w][p][f] = sum_j AinvT[w][p][j] C[f][j] = (C A^-1)[f][p]
        GemmArgs g;
        g.A = wd.AinvT[spin]; g.lda = s.nsp[spin]; g.strideA = (long)s.nsp[spin] * s.nsp[spin];
        g.B = s.Cplain[spin]; g.ldb = s.nsp[spin]; g.strideB = 0;   // the same coefficients for every walker
        g.C = Mt; g.ldc = s.nbp; g.strideC = (long)s.nsp[spin] * s.nbp;
        g.M = s.nsp[spin]; g.N = s.nbp; g.K = s.nsp[spin];
        cudaError_t e = gemm_f64_launch<CfgY128>(g, wd.W, EpiStore{}, st);
        COUNT_LAUNCH();
        if (e != cudaSuccess) return e;
    }
    if (s.ns[spin] > 0 || spin == 0) {
        k_dlogpsi<<<dim3(s.n_atoms, wd.W), 128, 0, st>>>(s, wd, spin, Mt, acc, spin == 0 ? 1 : 0);
        COUNT_LAUNCH();
    }
    return cudaGetLastError();
}

// Row f2, both halves.  Scratch (caller's): Mt, Nt [W][nsp_max][nbp]; Bm, U, XT [W][nsp_max^2]; fg [W][ne][8].
// acc_E [W][n_atoms][3] += dE_L/dR_a;  acc_psi (may be null) += d ln|Psi|/dR_a.  Both zeroed by the caller.
cudaError_t launch_forces(const SysDev& s, const WalkDev& wd, double* Mt, double* Nt, double* Bm, double* U, double* XT, double* fg,
                          double* acc_E, double* acc_psi, cudaStream_t st) {
    const long nsm = s.nsp[0] > s.nsp[1] ? s.nsp[0] : s.nsp[1];
    cudaError_t e = cudaMemsetAsync(Bm, 0, (size_t)2 * wd.W * nsm * nsm * 8, st);   // both spins: [2][W][nsm^2]
    if (e != cudaSuccess) return e;
    double* Bsp[2] = {Bm, Bm + (long)wd.W * nsm * nsm};
    k_force_prep<<<dim3((s.ne + 7) / 8, wd.W), 256, 0, st>>>(s, wd, fg, Bsp[0], Bsp[1]);
    COUNT_LAUNCH();
    for (int sp = 0; sp < 2; sp++) {
        const int nsp = s.nsp[sp];
        const long mat = (long)nsp * nsp;
        if (s.ns[sp] > 0) {
            GemmArgs g;
            // Mt[w][p][f] = sum_j AinvT[w][p][j] C[f][j] = (C A^-1)[f][p]
            g.A = wd.AinvT[sp]; g.lda = nsp; g.strideA = mat;
            g.B = s.Cplain[sp]; g.ldb = nsp; g.strideB = 0;
            g.C = Mt; g.ldc = s.nbp; g.strideC = (long)nsp * s.nbp;
            g.M = nsp; g.N = s.nbp; g.K = nsp;
            e = gemm_f64_launch<CfgY128>(g, wd.W, EpiStore{}, st);
            COUNT_LAUNCH();
            if (e != cudaSuccess) return e;
            // U[p][i] = sum_k AinvT[p][k] B[i][k]
            g.B = Bsp[sp]; g.ldb = nsp; g.strideB = mat;
            g.C = U; g.ldc = nsp; g.strideC = mat;
            g.N = nsp;
            e = gemm_f64_launch<CfgY128>(g, wd.W, EpiStore{}, st);
            COUNT_LAUNCH();
            if (e != cudaSuccess) return e;
            // XT[p][j] = sum_i U[p][i] AinvT[i][j] = X[j][p]
            g.A = U; g.B = wd.AinvT[sp]; g.C = XT;
            e = gemm_f64_launch<CfgUpd>(g, wd.W, EpiStore{}, st);
            COUNT_LAUNCH();
            if (e != cudaSuccess) return e;
            // Nt[w][p][f] = sum_j XT[w][p][j] C[f][j] = (C X)[f][p]
            g.A = XT;
            g.B = s.Cplain[sp]; g.ldb = nsp; g.strideB = 0;
            g.C = Nt; g.ldc = s.nbp; g.strideC = (long)nsp * s.nbp;
            g.N = s.nbp;
            e = gemm_f64_launch<CfgY128>(g, wd.W, EpiStore{}, st);
            COUNT_LAUNCH();
            if (e != cudaSuccess) return e;
        }
        if (s.ns[sp] > 0 || sp == 0) {
            k_deloc<<<dim3(s.n_atoms, wd.W), 128, 0, st>>>(s, wd, sp, Mt, Nt, fg, acc_E, acc_psi, sp == 0 ? 1 : 0);
            COUNT_LAUNCH();
        }
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// row f3: non-local pseudopotential energy (nlpp_kernels.cuh).  Two phases because the number of (electron, atom) pairs
// inside the cut-offs is data: nl_pairs_count leaves the offsets on the device (the host reads the total), nl_evaluate
// runs the points through basis values -> contraction -> ratios in chunks of 5 W points (the sweep's own Phi / V buffers).
cudaError_t launch_nl_count(const SysDev& s, const WalkDev& wd, const NlArgs& a, cudaStream_t st) {
    const long n = (long)wd.W * a.ns;
    if (n == 0) return cudaMemsetAsync(a.cnt, 0, 4, st);
    k_nl_count<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(s, wd, a);
    COUNT_LAUNCH();
    k_nl_scan<<<1, 1024, 0, st>>>(a.cnt, n);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
cudaError_t launch_nl_evaluate(const SysDev& s, const WalkDev& wd, const NlArgs& a, int n_pairs, int n_sm, unsigned* mo_epoch, double* vnl,
                               cudaStream_t st) {
    const long n = (long)wd.W * a.ns;
    if (n_pairs > 0) {
        k_nl_fill<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(s, wd, a);
        COUNT_LAUNCH();
        const long npts = 12L * n_pairs;
        k_nl_points<<<(unsigned)((npts + 255) / 256), 256, 0, st>>>(s, wd, a, n_pairs);
        COUNT_LAUNCH();
        const long chunk = 5L * wd.W;
        for (long p0 = 0; p0 < npts; p0 += chunk) {
            const int m = (int)(npts - p0 < chunk ? npts - p0 : chunk);
            cudaError_t e = launch_basis_values(s, a.pts + 3 * p0, m, wd.Phi, st);
            if (e != cudaSuccess) return e;
            e = launch_mo(s, a.spin, wd.Phi, m, wd.V, wd.ldv, wd.mo_ws, wd.mo_flags, mo_grid_for(s, a.spin, m, n_sm), ++*mo_epoch, nullptr, st);
            if (e != cudaSuccess) return e;
            k_nl_ratio<<<m, NL_RATIO_THREADS, 0, st>>>(s, wd, a, p0, m, wd.V);
            COUNT_LAUNCH();
        }
    }
    if (n > 0) {
        k_nl_reduce<<<wd.W, 256, 0, st>>>(wd, a, vnl);
        COUNT_LAUNCH();
    }
    return cudaGetLastError();
}

// the generator of k_step / k_sweep_small on caller-chosen counters and keys (cross-check against an independent
// implementation in the tests): in [n][6] = counter words 0..3, key words 0..1; out [n][4]
__global__ void k_philox_words(int n, const uint32_t* __restrict__ in, uint32_t* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t o[4];
    philox4x32_10(in[6 * i], in[6 * i + 1], in[6 * i + 2], in[6 * i + 3], in[6 * i + 4], in[6 * i + 5], o);
    out[4 * i] = o[0]; out[4 * i + 1] = o[1]; out[4 * i + 2] = o[2]; out[4 * i + 3] = o[3];
}
cudaError_t launch_philox_words(int n, const uint32_t* in, uint32_t* out, cudaStream_t st) {
    k_philox_words<<<(n + 255) / 256, 256, 0, st>>>(n, in, out);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

uint64_t launch_count() { return g_launches; }

}  // namespace qmc
