// qmc_kernels.cu -- the CUDA kernels of the batched electron move (sm_100a) and their launchers.
// Rows a1-a9 of SURVEY.md 8(a); formulas follow BASELINE.json north_star / DESIGN.md "Readings".
#include "qmc_kernels.cuh"

#include <math.h>

#include "gemm_f64.cuh"
#include "mo_streamk.cuh"

#ifndef QMC_UPD_BM
#define QMC_UPD_BM 128
#define QMC_UPD_BN 64
#define QMC_UPD_STAGES 2
#endif
#ifndef QMC_Y_STAGES
#define QMC_Y_STAGES 3
#endif

namespace qmc {

thread_local uint64_t g_launches = 0;
#define COUNT_LAUNCH() (++g_launches)

// ------------------------------------------------------------------------------------------------
// block reductions (fixed shape -> deterministic): NV sums at once over a block of NT threads
template <int NT, int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* red /* [NV * NT/32] */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NV; i++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    }
    __syncthreads();  // protect red from a previous use
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NV; i++) red[i * (NT / 32) + warp] = v[i];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; i++) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < NT / 32; k++) s += red[i * (NT / 32) + k];
        v[i] = s;
    }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------------
// Philox4x32-10, key = (seed lo, seed hi), counter = (walker, step, electron, block)   [reading A11]
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; r++) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ double u01(uint32_t we, uint32_t wo) {
    unsigned long long x = ((unsigned long long)we << 32) | (unsigned long long)wo;
    return (double)(2ull * (x >> 12) + 1ull) * 0x1.0p-53;  // odd integer * 2^-53: exact, in (0,1)
}

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

constexpr int BASIS_THREADS = 256;
constexpr int BASIS_MAXPT = (MO_BM + 4) / 5 + 1;  // points that can touch one 128-row tile (27)

// Work items are (point, shell) pairs, ordered s-shells | p-shells | d-shells of the k-block, so a warp mixes
// shell types only at the two boundaries (no divergence in the angular code elsewhere) and all 256 threads
// stay busy for the same number of passes.  The radial triple (three FP64 exp per pair -- the expensive part,
// issued as three independent chains) is computed once per shell and used from registers by its 2l+1 functions.
__global__ void __launch_bounds__(BASIS_THREADS, 4) k_basis(SysDev s, const double* __restrict__ pts, int n_points, double* __restrict__ out) {
    __shared__ __align__(128) double tile[MO_A_STAGE];  // [128][36]
    __shared__ double spt[3 * BASIS_MAXPT + 3];
    const int kb = blockIdx.x, tm = blockIdx.y, tid = threadIdx.x;
    const int row_lo = tm * MO_BM;
    const int pt_lo = row_lo / 5;
    int pt_hi = (row_lo + MO_BM + 4) / 5;
    if (pt_hi > n_points) pt_hi = n_points;
    const int npt = pt_hi - pt_lo;
    const int f_lo = kb * MO_BK;
    if (row_lo + MO_BM <= 5 * n_points && f_lo + MO_BK <= s.n_basis) {
        // every (row, function) of the tile gets written below: only the 4 padding columns need zeros
        for (int i = tid; i < MO_BM * 2; i += BASIS_THREADS)
            reinterpret_cast<double2*>(tile + (i >> 1) * MO_ALD + MO_BK)[i & 1] = make_double2(0.0, 0.0);
    } else {
        for (int i = tid; i < MO_A_STAGE / 2; i += BASIS_THREADS) reinterpret_cast<double2*>(tile)[i] = make_double2(0.0, 0.0);
    }
    if (tid < 3 * npt) spt[tid] = pts[3 * pt_lo + tid];
    __syncthreads();
    const int4 cnt = s.kb_counts[kb];  // x, y, z = number of s, p, d shells; w = offset of this block's list
    const KbShell* __restrict__ list = s.kb_list + cnt.w;
    const int r_base = pt_lo * 5 - row_lo;
    const int n0 = npt * cnt.x, n1 = n0 + npt * cnt.y, n2 = n1 + npt * cnt.z;
    for (int q = tid; q < n2; q += BASIS_THREADS) {
        int L, qq, c, base;
        if (q < n0) { L = 0; qq = q; c = cnt.x; base = 0; }
        else if (q < n1) { L = 1; qq = q - n0; c = cnt.y; base = cnt.x; }
        else { L = 2; qq = q - n1; c = cnt.z; base = cnt.x + cnt.y; }
        const int pi = qq / c;
        const KbShell rec = list[base + qq - pi * c];
        const double x = spt[3 * pi] - rec.x, y = spt[3 * pi + 1] - rec.y, z = spt[3 * pi + 2] - rec.z;
        const double t = x * x + y * y + z * z;
        // accumulation order p = 0, 1, 2, ... as in the definition of g, g', g''
        const double e0 = rec.c[0] * exp(-rec.a[0] * t), e1 = rec.c[1] * exp(-rec.a[1] * t), e2 = rec.c[2] * exp(-rec.a[2] * t);
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
        const int r0 = r_base + pi * 5;  // local row of the value component (may be < 0 or > 123)
        const int c0 = rec.f0 - f_lo;
        const double lapfac = (double)(4 * L + 6) * g1 + 4.0 * t * g2;
        const double tg1 = 2.0 * g1;
        auto emit = [&](int m, double S, double Sx, double Sy, double Sz) {
            const int col = c0 + m;
            if (col < 0 || col >= MO_BK) return;
            const double v[5] = {S * g, g * Sx + tg1 * S * x, g * Sy + tg1 * S * y, g * Sz + tg1 * S * z, S * lapfac};
#pragma unroll
            for (int k = 0; k < 5; k++)
                if (r0 + k >= 0 && r0 + k < MO_BM) tile[(r0 + k) * MO_ALD + col] = v[k];
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
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // generic-proxy smem writes -> visible to the TMA engine
    __syncthreads();
    if (tid == 0) {
        bulk_s2g(out + ((long)tm * s.kb + kb) * MO_A_STAGE, tile, MO_A_STAGE * sizeof(double));
        asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory");  // smem must outlive the read
    }
}

cudaError_t launch_basis(const SysDev& s, const double* pts, int n_points, double* PhiT, cudaStream_t st) {
    if (n_points == 0) return cudaSuccess;
    dim3 grid(s.kb, (5 * n_points + MO_BM - 1) / MO_BM);
    k_basis<<<grid, BASIS_THREADS, 0, st>>>(s, pts, n_points, PhiT);
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

cudaError_t launch_mo(const SysDev& s, int spin, const double* PhiT, int rows, double* V, long ldv, double* ws, unsigned* flags,
                      int grid, unsigned epoch, cudaStream_t st) {
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_mo_streamk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MO_SMEM_BYTES);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    MoArgs g;
    g.PhiT = PhiT; g.CT = s.CT[spin]; g.V = V; g.ldv = ldv;
    g.M = rows; g.N = s.nsp[spin];
    g.MT = (rows + MO_BM - 1) / MO_BM; g.NT = s.nt[spin]; g.KB = s.kb;
    g.ws = ws; g.flags = flags; g.epoch = epoch;
    if (grid < 1) return cudaSuccess;
    k_mo_streamk<<<grid, MO_THREADS, MO_SMEM_BYTES, st>>>(g);
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Pade Jastrow pieces
__device__ __forceinline__ double pade_u(double a, double b, double r) { return a * r / (1.0 + b * r); }
__device__ __forceinline__ double pade_du(double a, double b, double r) { double q = 1.0 + b * r; return a / (q * q); }
__device__ __forceinline__ double pade_d2u(double a, double b, double r) { double q = 1.0 + b * r; return -2.0 * a * b / (q * q * q); }

// partner k of electron e: k < ne electrons (skip k == e), then atoms
struct Partner { double x, y, z, a, b; bool ok; };
__device__ __forceinline__ Partner partner(const SysDev& s, const double* __restrict__ Rw, int nep, int e, int k) {
    Partner P;
    if (k < s.ne) {
        P.x = Rw[k]; P.y = Rw[nep + k]; P.z = Rw[2 * nep + k];
        const bool same = (k < s.ns[0]) == (e < s.ns[0]);
        P.a = same ? s.a_para : s.a_anti;
        P.b = s.b_ee;
        P.ok = (k != e);
    } else {
        const int I = k - s.ne;
        P.x = s.atom_xyz[3 * I]; P.y = s.atom_xyz[3 * I + 1]; P.z = s.atom_xyz[3 * I + 2];
        P.a = -s.atom_Z[I];
        P.b = s.b_en;
        P.ok = true;
    }
    return P;
}

// ------------------------------------------------------------------------------------------------
// a1 + a2 + a6: effective inverse column, drift, Philox proposal, Jastrow ratio and gradient at r'.
// One CTA of 512 threads per walker.  The two streaming passes over the delay window (b = Vbuf a_p, then
// x = a_p - Wbuf^T c) are HBM-bound GEMVs: every thread keeps 8 independent 16-byte loads in flight.
//                                                                               [north_star items 3, 4]
constexpr int PT = 512;
constexpr int PW = PT / 32;

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

// dot products of row[0..n) with xs[0..n) (n % 2 == 0), one warp, 8 loads in flight per lane
__device__ __forceinline__ double warp_dot(const double* __restrict__ row, const double* xs, int n, int lane) {
    double acc = 0.0;
    const int n2 = n >> 1;
    int j = lane;
    for (; j + 7 * 32 < n2; j += 8 * 32) {
        double2 a[8];
#pragma unroll
        for (int u = 0; u < 8; u++) a[u] = ldg2(row + 2 * (j + u * 32));
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const double2 x = *reinterpret_cast<const double2*>(xs + 2 * (j + u * 32));
            acc += a[u].x * x.x + a[u].y * x.y;
        }
    }
    for (; j < n2; j += 32) {
        const double2 a = ldg2(row + 2 * j);
        const double2 x = *reinterpret_cast<const double2*>(xs + 2 * j);
        acc += a.x * x.x + a.y * x.y;
    }
    return warp_sum(acc);
}

__global__ void __launch_bounds__(PT, 2) k_propose(SysDev s, WalkDev wd, int spin, int p, int e, uint32_t step, double tau,
                                                double sqrt_tau) {
    extern __shared__ __align__(16) double sm[];
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nsp = s.nsp[spin], kp = wd.kp, nep = wd.nep;
    const int kps = kp + 1;            // padded row stride of the S^-1 copy (conflict-free column walks)
    double* xs = sm;                   // [nsp]
    double* bs = xs + nsp;             // [kp]
    double* cs = bs + kp;              // [kp]
    double* red = cs + kp;             // [8 * PW]
    double* bc = red + 8 * PW;         // [4] broadcast
    double* Ss = bc + 4;               // [kp][kp + 1]
    const double* arow = wd.AinvT[spin] + ((long)w * nsp + p) * nsp;
    const int m = wd.mcount[w];
    for (int j = tid; j < nsp / 2; j += PT) reinterpret_cast<double2*>(xs)[j] = ldg2(arow + 2 * j);
    if (m > 0) {
        const double* Si = wd.SinvT + (long)w * kp * kp;
        for (int idx = tid; idx < m * kp; idx += PT) {
            const int l = idx / kp, n = idx - l * kp;
            if (n < m) Ss[l * kps + n] = Si[idx];
        }
    }
    __syncthreads();
    if (m > 0) {
        // b_n = v_n . a_p ;  c = S^-1 b ;  x = a_p - Wbuf^T c     (effective column of the delayed inverse)
        const double* Vb = wd.Vbuf + (long)w * kp * nsp;
        const double* Wb = wd.Wbuf + (long)w * kp * nsp;
        for (int n = warp; n < m; n += PW) {
            const double acc = warp_dot(Vb + (long)n * nsp, xs, nsp, lane);
            if (lane == 0) bs[n] = acc;
        }
        __syncthreads();
        for (int n = tid; n < m; n += PT) {
            double acc = 0.0;
            for (int l = 0; l < m; l++) acc += Ss[l * kps + n] * bs[l];
            cs[n] = acc;
            wd.cvec[(long)w * kp + n] = acc;
        }
        __syncthreads();
        for (int j = tid; j < nsp / 2; j += PT) {
            double2 acc = reinterpret_cast<double2*>(xs)[j];
            int l = 0;
            for (; l + 8 <= m; l += 8) {
                double2 wv[8];
#pragma unroll
                for (int u = 0; u < 8; u++) wv[u] = ldg2(Wb + (long)(l + u) * nsp + 2 * j);
#pragma unroll
                for (int u = 0; u < 8; u++) { acc.x -= cs[l + u] * wv[u].x; acc.y -= cs[l + u] * wv[u].y; }
            }
            for (; l < m; l++) {
                const double2 wv = ldg2(Wb + (long)l * nsp + 2 * j);
                acc.x -= cs[l] * wv.x; acc.y -= cs[l] * wv.y;
            }
            reinterpret_cast<double2*>(xs)[j] = acc;
        }
        __syncthreads();
    }
    double* xcol = wd.xcol + (long)w * nsp;
    for (int j = tid; j < nsp / 2; j += PT) reinterpret_cast<double2*>(xcol)[j] = reinterpret_cast<double2*>(xs)[j];

    // drift: determinant part from the cached gradient rows, Jastrow part by direct sums
    const double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    const double* Rw = wd.R + (long)w * 3 * nep;
    const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
    double acc6[6] = {0, 0, 0, 0, 0, 0};
    for (int j = tid; j < nsp / 2; j += PT) {
        const double2 xj = reinterpret_cast<double2*>(xs)[j];
        const double2 o1 = ldg2(orb + nsp + 2 * j), o2 = ldg2(orb + 2 * nsp + 2 * j), o3 = ldg2(orb + 3 * nsp + 2 * j);
        acc6[0] += o1.x * xj.x + o1.y * xj.y;
        acc6[1] += o2.x * xj.x + o2.y * xj.y;
        acc6[2] += o3.x * xj.x + o3.y * xj.y;
    }
    const int npart = s.ne + s.n_atoms;
    for (int k = tid; k < npart; k += PT) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double du = pade_du(P.a, P.b, r);
            acc6[3] += du * dx / r;
            acc6[4] += du * dy / r;
            acc6[5] += du * dz / r;
        }
    }
    block_sum<PT, 6>(acc6, red);
    if (tid == 0) {
        const double Gx = acc6[0] + acc6[3], Gy = acc6[1] + acc6[4], Gz = acc6[2] + acc6[5];
        const uint32_t wid = wd.first_walker + (uint32_t)w;
        const uint32_t k0 = (uint32_t)(wd.seed & 0xFFFFFFFFull), k1 = (uint32_t)(wd.seed >> 32);
        uint32_t o[4];
        philox4x32_10(wid, step, (uint32_t)e, 0u, k0, k1, o);
        const double U1 = u01(o[0], o[1]), U2 = u01(o[2], o[3]);
        philox4x32_10(wid, step, (uint32_t)e, 1u, k0, k1, o);
        const double U3 = u01(o[0], o[1]), U4 = u01(o[2], o[3]);
        philox4x32_10(wid, step, (uint32_t)e, 2u, k0, k1, o);
        const double U5 = u01(o[0], o[1]);
        const double TWO_PI = 6.283185307179586;
        const double r1 = sqrt(-2.0 * log(U1)), r2 = sqrt(-2.0 * log(U3));
        const double chx = r1 * cos(TWO_PI * U2), chy = r1 * sin(TWO_PI * U2), chz = r2 * cos(TWO_PI * U4);
        const double qx = rx + tau * Gx + sqrt_tau * chx;
        const double qy = ry + tau * Gy + sqrt_tau * chy;
        const double qz = rz + tau * Gz + sqrt_tau * chz;
        wd.rp[3 * w] = qx; wd.rp[3 * w + 1] = qy; wd.rp[3 * w + 2] = qz;
        wd.G[3 * w] = Gx; wd.G[3 * w + 1] = Gy; wd.G[3 * w + 2] = Gz;
        wd.u[w] = U5;
        bc[0] = qx; bc[1] = qy; bc[2] = qz;
    }
    __syncthreads();
    const double qx = bc[0], qy = bc[1], qz = bc[2];
    // Jastrow ratio (term by term) and gradient at r'
    double acc4[4] = {0, 0, 0, 0};
    for (int k = tid; k < npart; k += PT) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double ex = qx - P.x, ey = qy - P.y, ez = qz - P.z;
            const double r_old = sqrt(dx * dx + dy * dy + dz * dz);
            const double r_new = sqrt(ex * ex + ey * ey + ez * ez);
            acc4[0] += pade_u(P.a, P.b, r_new) - pade_u(P.a, P.b, r_old);
            const double du = pade_du(P.a, P.b, r_new);
            acc4[1] += du * ex / r_new;
            acc4[2] += du * ey / r_new;
            acc4[3] += du * ez / r_new;
        }
    }
    block_sum<PT, 4>(acc4, red);
    if (tid == 0) {
        wd.dJ[w] = acc4[0];
        wd.gJn[3 * w] = acc4[1]; wd.gJn[3 * w + 1] = acc4[2]; wd.gJn[3 * w + 2] = acc4[3];
    }
}

size_t propose_smem(const SysDev& s, const WalkDev& wd, int spin) {
    return (size_t)(s.nsp[spin] + 2 * wd.kp + 8 * PW + 4 + wd.kp * (wd.kp + 1)) * sizeof(double);
}

cudaError_t launch_propose(const SysDev& s, const WalkDev& wd, int spin, int p, int e, uint32_t step, double tau, cudaStream_t st) {
    static size_t configured = 48 * 1024;
    const size_t smem = propose_smem(s, wd, spin);
    if (smem > configured) {
        cudaError_t er = cudaFuncSetAttribute(k_propose, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (er != cudaSuccess) return er;
        configured = smem;
    }
    k_propose<<<wd.W, PT, smem, st>>>(s, wd, spin, p, e, step, tau, sqrt(tau));
    COUNT_LAUNCH();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a5 + a7: determinant ratio and gradient from the effective column, accept/reject, commit.
// One CTA per walker.  commit == 0 evaluates everything but changes no state (stage timing).
__global__ void __launch_bounds__(PT, 2) k_accept(SysDev s, WalkDev wd, int spin, int p, int e, long log_off, double tau, int commit) {
    extern __shared__ __align__(16) double sm[];
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nsp = s.nsp[spin], kp = wd.kp, nep = wd.nep;
    const int kps = kp + 1;
    double* vs = sm;                   // [nsp] value row of the proposed position
    double* rs = vs + nsp;             // [kp]
    double* ts = rs + kp;              // [kp]
    double* cs = ts + kp;              // [kp]
    double* red = cs + kp;             // [8 * PW]
    double* bc = red + 8 * PW;         // [4]
    double* Ss = bc + 4;               // [kp][kp + 1]
    const double* v = wd.V + (long)w * 5 * wd.ldv;
    const double* xcol = wd.xcol + (long)w * nsp;
    double a4[4] = {0, 0, 0, 0};
    for (int j = tid; j < nsp / 2; j += PT) {
        const double2 xj = ldg2(xcol + 2 * j);
        const double2 v0 = ldg2(v + 2 * j), v1 = ldg2(v + wd.ldv + 2 * j), v2 = ldg2(v + 2 * wd.ldv + 2 * j), v3 = ldg2(v + 3 * wd.ldv + 2 * j);
        reinterpret_cast<double2*>(vs)[j] = v0;
        a4[0] += v0.x * xj.x + v0.y * xj.y;
        a4[1] += v1.x * xj.x + v1.y * xj.y;
        a4[2] += v2.x * xj.x + v2.y * xj.y;
        a4[3] += v3.x * xj.x + v3.y * xj.y;
    }
    block_sum<PT, 4>(a4, red);
    const double rho = a4[0];
    if (tid == 0) {
        double* Rw = wd.R + (long)w * 3 * nep;
        const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
        const double qx = wd.rp[3 * w], qy = wd.rp[3 * w + 1], qz = wd.rp[3 * w + 2];
        const double Gx = wd.G[3 * w], Gy = wd.G[3 * w + 1], Gz = wd.G[3 * w + 2];
        const double u = wd.u[w], dJ = wd.dJ[w];
        unsigned bits = 0;
        double pacc = 0.0, jr = 0.0;
        bool accept = false;
        if (fabs(rho) < 1e-12) bits |= 2u;
        if (rho > 0.0) {  // fixed node: reject rho_D <= 0 (A7); NaN fails the comparison and rejects
            const double Hx = a4[1] / rho + wd.gJn[3 * w], Hy = a4[2] / rho + wd.gJn[3 * w + 1], Hz = a4[3] / rho + wd.gJn[3 * w + 2];
            const double ax = qx - rx - tau * Gx, ay = qy - ry - tau * Gy, az = qz - rz - tau * Gz;
            const double cx = rx - qx - tau * Hx, cy = ry - qy - tau * Hy, cz = rz - qz - tau * Hz;
            const double fwd = ax * ax + ay * ay + az * az, rev = cx * cx + cy * cy + cz * cz;
            const double Delta = (fwd - rev) / (2.0 * tau);
            pacc = rho * rho * exp(2.0 * dJ + Delta);  // A25: linear domain, one exp
            jr = rho * exp(dJ);
            if (fabs(u - pacc) < 1e-12) bits |= 2u;
            accept = (u < pacc);
        }
        const bool nonfinite = isnan(rho) || isnan(pacc);
        if (nonfinite) { bits |= 4u; accept = false; }
        if (accept) bits |= 1u;
        if (commit) {
            wd.bits[log_off + w] = (uint8_t)bits;
            if (wd.ratio_log) { wd.ratio_log[log_off + w] = jr; wd.pacc_log[log_off + w] = pacc; }
            atomicAdd(&wd.stats[0], 1ull);
            if (accept) atomicAdd(&wd.stats[1], 1ull);
            if (bits & 2u) atomicAdd(&wd.stats[2], 1ull);
            if (nonfinite) { atomicAdd(&wd.stats[3], 1ull); wd.flags[w] = 1u; }
            if (accept) {
                Rw[e] = qx; Rw[nep + e] = qy; Rw[2 * nep + e] = qz;
                wd.logpsi[w] += log(rho) + dJ;
            }
        }
        bc[0] = (accept && commit) ? 1.0 : 0.0;
    }
    __syncthreads();
    if (bc[0] == 0.0) return;
    // ---- commit: row caches, delay window (Vbuf, Wbuf, bordered update of S^-1)
    const int m = wd.mcount[w];
    double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    double* Vb = wd.Vbuf + (long)w * kp * nsp;
    double* Wb = wd.Wbuf + (long)w * kp * nsp;
    double* Si = wd.SinvT + (long)w * kp * kp;
    const double* arow = wd.AinvT[spin] + ((long)w * nsp + p) * nsp;
    // r_l = v . Wbuf[l]  (row m of S): the streaming pass, issued first
    for (int l = warp; l < m; l += PW) {
        const double acc = warp_dot(Wb + (long)l * nsp, vs, nsp, lane);
        if (lane == 0) rs[l] = acc;
    }
    for (int idx = tid; idx < m * kp; idx += PT) {
        const int l = idx / kp, n = idx - l * kp;
        if (n < m) Ss[l * kps + n] = Si[idx];
    }
    for (int n = tid; n < m; n += PT) cs[n] = wd.cvec[(long)w * kp + n];
    for (int j = tid; j < nsp / 2; j += PT) {
        const double2 a = ldg2(arow + 2 * j);
        const double2 v1 = ldg2(v + wd.ldv + 2 * j), v2 = ldg2(v + 2 * wd.ldv + 2 * j), v3 = ldg2(v + 3 * wd.ldv + 2 * j), v4 = ldg2(v + 4 * wd.ldv + 2 * j);
        const double2 v0 = reinterpret_cast<double2*>(vs)[j];
        reinterpret_cast<double2*>(orb)[j] = v0;
        reinterpret_cast<double2*>(orb + nsp)[j] = v1;
        reinterpret_cast<double2*>(orb + 2 * nsp)[j] = v2;
        reinterpret_cast<double2*>(orb + 3 * nsp)[j] = v3;
        reinterpret_cast<double2*>(orb + 4 * nsp)[j] = v4;
        reinterpret_cast<double2*>(Vb + (long)m * nsp)[j] = v0;
        reinterpret_cast<double2*>(Wb + (long)m * nsp)[j] = a;
    }
    __syncthreads();
    // t_l = sum_n r_n Sinv[n][l] = sum_n r_n SinvT[l][n]
    for (int l = tid; l < m; l += PT) {
        double acc = 0.0;
        for (int n = 0; n < m; n++) acc += rs[n] * Ss[l * kps + n];
        ts[l] = acc;
    }
    __syncthreads();
    const double sinv = 1.0 / rho;
    for (int idx = tid; idx < m * m; idx += PT) {
        const int l = idx / m, n = idx % m;
        Si[l * kp + n] = Ss[l * kps + n] + cs[n] * ts[l] * sinv;
    }
    for (int n = tid; n < m; n += PT) {
        Si[m * kp + n] = -cs[n] * sinv;
        Si[n * kp + m] = -ts[n] * sinv;
    }
    if (tid == 0) {
        Si[m * kp + m] = sinv;
        wd.plist[(long)w * kp + m] = p;
        wd.mcount[w] = m + 1;
    }
}

cudaError_t launch_accept(const SysDev& s, const WalkDev& wd, int spin, int p, int e, long log_off, double tau, int commit, cudaStream_t st) {
    static size_t configured = 48 * 1024;
    const size_t smem = (size_t)(s.nsp[spin] + 3 * wd.kp + 8 * PW + 4 + wd.kp * (wd.kp + 1)) * sizeof(double);
    if (smem > configured) {
        cudaError_t er = cudaFuncSetAttribute(k_accept, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (er != cudaSuccess) return er;
        configured = smem;
    }
    k_accept<<<wd.W, PT, smem, st>>>(s, wd, spin, p, e, log_off, tau, commit);
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
using CfgAcc = GemmCfg<QMC_UPD_BM, QMC_UPD_BN, 64, 32, false, QMC_UPD_STAGES>;  // flush update: several CTAs per SM

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

cudaError_t launch_flush(const SysDev& s, const WalkDev& wd, int spin, cudaStream_t st) {
    const int nsp = s.nsp[spin], kp = wd.kp;
    cudaError_t e;
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
__global__ void __launch_bounds__(256) k_eloc_elec(SysDev s, WalkDev wd) {
    const int w = blockIdx.y;
    const int e = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (e >= s.ne) return;
    const int spin = e < s.ns[0] ? 0 : 1, p = spin ? e - s.ns[0] : e;
    const int nsp = s.nsp[spin], nep = wd.nep;
    const double* arow = wd.AinvT[spin] + ((long)w * nsp + p) * nsp;
    const double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    double gx = 0, gy = 0, gz = 0, lp = 0;
    for (int j = lane; j < nsp; j += 32) {
        const double a = arow[j];
        gx += orb[nsp + j] * a;
        gy += orb[2 * nsp + j] * a;
        gz += orb[3 * nsp + j] * a;
        lp += orb[4 * nsp + j] * a;
    }
    const double* Rw = wd.R + (long)w * 3 * nep;
    const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
    double jx = 0, jy = 0, jz = 0, jl = 0, pot = 0;
    const int npart = s.ne + s.n_atoms;
    for (int k = lane; k < npart; k += 32) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double du = pade_du(P.a, P.b, r);
            jx += du * dx / r; jy += du * dy / r; jz += du * dz / r;
            jl += pade_d2u(P.a, P.b, r) + 2.0 * du / r;
            if (k >= s.ne) pot += P.a / r;          // P.a = -Z_I
            else if (k > e) pot += 1.0 / r;         // each pair once
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

cudaError_t launch_gj_inverse(double* Mall, long stride, int n, int ld, int batch, double* logdet, int* sign, int* status, cudaStream_t st) {
    if (n == 0 || batch == 0) return cudaSuccess;
    COUNT_LAUNCH();
    if (n >= 512) {
        constexpr int NT = 1024;
        size_t smem = (size_t)(2 * n + NT / 32) * sizeof(double) + (size_t)(NT / 32 + n) * sizeof(int);
        cudaFuncSetAttribute(k_gj_inverse<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
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
__global__ void k_tile_C(const double* __restrict__ in, int nb, int ns, double* __restrict__ CT, int kb) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)nb * ns) return;
    const int l = (int)(idx / ns), j = (int)(idx % ns);
    CT[cT_index(l, j, kb)] = in[idx];
}
cudaError_t launch_tile_C(const double* in, int nb, int ns, double* CT, int kb, cudaStream_t st) {
    long n = (long)nb * ns;
    if (n == 0) return cudaSuccess;
    k_tile_C<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, nb, ns, CT, kb);
    COUNT_LAUNCH();
    return cudaGetLastError();
}
__global__ void k_export_phi(const double* __restrict__ PhiT, long n_rows, int width, int kb, double* __restrict__ out) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_rows * width) return;
    out[idx] = PhiT[phiT_index(idx / width, (int)(idx % width), kb)];
}
cudaError_t launch_export_phi(const double* PhiT, long n_rows, int width, int kb, double* out, cudaStream_t st) {
    long n = n_rows * width;
    if (n == 0) return cudaSuccess;
    k_export_phi<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(PhiT, n_rows, width, kb, out);
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

uint64_t launch_count() { return g_launches; }

}  // namespace qmc
