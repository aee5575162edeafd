// step_kernel.cuh -- the per-walker part of one electron step: rows a5 + a7 (ratio, accept/reject, commit)
// of electron p fused with rows a1 + a2 + a6 (effective column, drift, Philox proposal, Jastrow) of electron
// p + 1, in ONE kernel, one CTA of 512 threads per walker.        [BASELINE.json north_star items 3, 4]
//
// Between the MO contraction of electron p and the basis evaluation of electron p + 1 everything a walker
// does is private to it, so the two halves share a launch; at the ends of a delay window (a flush sits in
// between) the same kernel runs with only one half enabled.
//
// The work is HBM-bound: per proposal the walker streams its delay window -- Wbuf for r = Wbuf v (commit),
// Vbuf for b = Vbuf a_p, Wbuf again for x = a_p - Wbuf^T c -- 8 KB rows at config 2.  The two dot-product
// passes run as ONE pass (a warp takes row l of both matrices), every lane keeping 8 independent 16-byte
// loads in flight; no block-wide barrier inside a pass.  (A TMA-bulk ring through shared memory was measured
// slower here: the per-batch barriers cost more than the registers the direct loads need.)
#pragma once
#include "device_utils.cuh"
#include "mo_streamk.cuh"  // mbarrier / bulk-copy wrappers
#include "qmc_internal.cuh"

namespace qmc {

// threads per walker: 512 for the large systems the kernel was tuned on (8 KB rows at config 2), 128 where a row of the
// inverse is at most 256 doubles -- there 512 threads would mostly wait at barriers, and four times as many CTAs fit an SM.
// lean: the crowd runs as two lanes whose step kernels share the SMs with the OTHER lane's persistent contraction
// (168 registers x 288 threads resident): 256 threads x 64 registers is what fits beside it.
__host__ __device__ inline int step_threads(int nsp, bool lean = false) { return nsp <= 256 ? 128 : (lean ? 256 : 512); }

// shared-memory carve-up (in doubles)
struct StepLayout {
    int xs, vs, as, c4, bs, cs, rs, ts, red, bc, total;
    __host__ __device__ StepLayout(int nsp, int kp, int PW /* warps per CTA */) {
        xs = 0; vs = xs + nsp; as = vs + nsp; c4 = as + nsp;
        bs = c4 + 32 * PW;   // c4: PT / 128 partial sums for each of 128 window rows
        cs = bs + kp + 1; rs = cs + kp + 1; ts = rs + kp + 1;
        red = ts + kp + 1; bc = red + 8 * PW; total = bc + 16;
    }
};
inline size_t step_smem_bytes(int nsp, int kp, bool lean = false) { return (size_t)StepLayout(nsp, kp, step_threads(nsp, lean) / 32).total * sizeof(double); }

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
// COH: the data may have been written earlier in the SAME launch (the window kernel of the mid-size path runs several
// electron steps per launch): read it through L2 (ld.global.cg), not through the non-coherent read-only path
template <bool COH>
__device__ __forceinline__ double2 ld2(const double* p) {
    return COH ? __ldcg(reinterpret_cast<const double2*>(p)) : __ldg(reinterpret_cast<const double2*>(p));
}

// The threads that work on one walker: a whole CTA (k_step) or a 128-thread group of a CTA (k_window), which then meets at
// a named barrier instead of __syncthreads.
struct CtaSync {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
template <int NT>
struct GroupSync {
    int id;   // named barrier 1..15
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;\n" ::"r"(id), "n"(NT) : "memory"); }
};
template <int NT, int NV, class Sync>
__device__ __forceinline__ void group_sum(double (&v)[NV], double* red /* [NV * NT/32] */, int tid, const Sync& sync) {
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int i = 0; i < NV; i++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    }
    sync();  // protect red from a previous use
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NV; i++) red[i * (NT / 32) + warp] = v[i];
    }
    sync();
#pragma unroll
    for (int i = 0; i < NV; i++) {
        double sacc = 0.0;
#pragma unroll
        for (int k = 0; k < NT / 32; k++) sacc += red[i * (NT / 32) + k];
        v[i] = sacc;
    }
}

// One warp: accA = rowA . vecA and (if rowB) accB = rowB . vecB over n2 double2's; rows in HBM (read-only path),
// vectors in shared memory; 8 independent 16-byte loads in flight per lane.
template <bool COH>
__device__ __forceinline__ void warp_dot2(const double* __restrict__ rowA, const double* vecA, const double* __restrict__ rowB, const double* vecB,
                                          int n2, int lane, double& accA, double& accB) {
    const double2* xa = reinterpret_cast<const double2*>(vecA);
    const double2* xb = reinterpret_cast<const double2*>(vecB);
    double sa = 0.0, sb = 0.0;
    int j = lane;
    if (rowB) {
        for (; j + 3 * 32 < n2; j += 4 * 32) {
            double2 a[4], b[4];
#pragma unroll
            for (int u = 0; u < 4; u++) { a[u] = ld2<COH>(rowA + 2 * (j + u * 32)); b[u] = ld2<COH>(rowB + 2 * (j + u * 32)); }
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const double2 x = xa[j + u * 32], y = xb[j + u * 32];
                sa += a[u].x * x.x + a[u].y * x.y;
                sb += b[u].x * y.x + b[u].y * y.y;
            }
        }
        for (; j < n2; j += 32) {
            const double2 a = ld2<COH>(rowA + 2 * j), b = ld2<COH>(rowB + 2 * j), x = xa[j], y = xb[j];
            sa += a.x * x.x + a.y * x.y;
            sb += b.x * y.x + b.y * y.y;
        }
    } else {
        for (; j + 7 * 32 < n2; j += 8 * 32) {
            double2 a[8];
#pragma unroll
            for (int u = 0; u < 8; u++) a[u] = ld2<COH>(rowA + 2 * (j + u * 32));
#pragma unroll
            for (int u = 0; u < 8; u++) {
                const double2 x = xa[j + u * 32];
                sa += a[u].x * x.x + a[u].y * x.y;
            }
        }
        for (; j < n2; j += 32) {
            const double2 a = ld2<COH>(rowA + 2 * j), x = xa[j];
            sa += a.x * x.x + a.y * x.y;
        }
    }
    accA = warp_sum(sa);
    accB = warp_sum(sb);
}

// Short rows (n2 <= 128 double2: at most 256 orbitals per spin): a warp takes R window rows at once -- rows l, l + dl,
// ... -- so that R x 2 loads are in flight per lane instead of two; one row at a time is one memory latency per row.
template <bool COH, int R>
__device__ __forceinline__ void warp_dot2_rows(const double* __restrict__ rowA, const double* vecA, const double* __restrict__ rowB, const double* vecB,
                                               long row_stride, int n_rows, int n2, int lane, double (&accA)[R], double (&accB)[R]) {
    const double2* xa = reinterpret_cast<const double2*>(vecA);
    const double2* xb = reinterpret_cast<const double2*>(vecB);
    double sa[R], sb[R];
#pragma unroll
    for (int r = 0; r < R; r++) sa[r] = sb[r] = 0.0;
    for (int j = lane; j < n2; j += 32) {
        double2 a[R], b[R];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const long o = (r < n_rows ? r : 0) * row_stride + 2 * j;
            a[r] = rowA ? ld2<COH>(rowA + o) : make_double2(0.0, 0.0);
            b[r] = rowB ? ld2<COH>(rowB + o) : make_double2(0.0, 0.0);
        }
        const double2 x = xa[j], y = xb[j];
#pragma unroll
        for (int r = 0; r < R; r++) {
            sa[r] += a[r].x * x.x + a[r].y * x.y;
            sb[r] += b[r].x * y.x + b[r].y * y.y;
        }
    }
#pragma unroll
    for (int r = 0; r < R; r++) { accA[r] = warp_sum(sa[r]); accB[r] = warp_sum(sb[r]); }
}

// Drift limiter of the DMC generation (row f1, reading A28; Umrigar-Nightingale-Runge 1993 eq. 35 with one constant a):
// vbar = v (-1 + sqrt(1 + 2 a v^2 tau)) / (a v^2 tau), evaluated as v * 2 / (1 + sqrt(1 + 2x)), x = a v^2 tau (the same
// number without the cancellation at small x).  a <= 0: off (reading A6).
__device__ __forceinline__ void limit_drift(double& gx, double& gy, double& gz, double lim_a, double tau) {
    if (!(lim_a > 0.0)) return;
    const double v2 = gx * gx + gy * gy + gz * gz;
    const double x = lim_a * v2 * tau;
    const double sc = 2.0 / (1.0 + sqrt(1.0 + 2.0 * x));
    gx *= sc; gy *= sc; gz *= sc;
}

// The body works on walker w with the PT threads tid = 0..PT-1 that `sync` joins, in their shared memory `sm`
// (StepLayout(nsp, kp, PT / 32).total doubles).  Every branch that leaves it is uniform over those threads.
template <int PT, bool COH, class Sync>
__device__ __forceinline__ void step_body(const SysDev& s, const WalkDev& wd, int w, int tid, double* sm, const Sync& sync, int spin, int p_acc,
                                          int p_prop, long log_off, uint32_t step, double tau, double sqrt_tau, int commit) {
    const int lane = tid & 31, warp = tid >> 5;
    const int nsp = s.nsp[spin], n2 = nsp >> 1, kp = wd.kp, nep = wd.nep;
    const int e0 = spin == 0 ? 0 : s.ns[0];
    constexpr int PW = PT / 32;
    const StepLayout L(nsp, kp, PW);
    double *xs = sm + L.xs, *vs = sm + L.vs, *as = sm + L.as, *c4 = sm + L.c4;
    double *bs = sm + L.bs, *cs = sm + L.cs, *rs = sm + L.rs, *ts = sm + L.ts, *red = sm + L.red, *bc = sm + L.bc;
    double* Rw = wd.R + (long)w * 3 * nep;
    double* Vb = wd.Vbuf + (long)w * kp * nsp;
    double* Wb = wd.Wbuf + (long)w * kp * nsp;
    double* Si = wd.SinvT + (long)w * kp * kp;
    const int m_old = wd.mcount[w];  // window rows written by earlier kernels (safe for the read-only path)
    bool accepted = false;
    double rho = 1.0;

    if (p_prop >= 0) {
        if (warp == 1 && lane < 3) {
            // the random numbers of the proposal depend on nothing: one Philox block per lane, off the critical path
            const uint32_t wid = wd.first_walker + (uint32_t)w;
            const uint32_t k0 = (uint32_t)(wd.seed & 0xFFFFFFFFull), k1 = (uint32_t)(wd.seed >> 32);
            uint32_t o[4];
            philox4x32_10(wid, step, (uint32_t)(e0 + p_prop), (uint32_t)lane, k0, k1, o);
            const double Ua = u01(o[0], o[1]), Ub = u01(o[2], o[3]);
            const double TWO_PI = 6.283185307179586;
            if (lane == 0) { const double r1 = sqrt(-2.0 * log(Ua)); bc[4] = r1 * cos(TWO_PI * Ub); bc[5] = r1 * sin(TWO_PI * Ub); }
            if (lane == 1) { const double r2 = sqrt(-2.0 * log(Ua)); bc[6] = r2 * cos(TWO_PI * Ub); }
            if (lane == 2) bc[7] = Ua;
        }
        const double* arow = wd.AinvT[spin] + ((long)w * nsp + p_prop) * nsp;
        for (int j = tid; j < n2; j += PT) reinterpret_cast<double2*>(xs)[j] = ldg2(arow + 2 * j);
    }

    // =================================================================== a5 + a7 for electron p_acc
    const double* v = wd.V + (long)w * 5 * wd.ldv;
    if (p_acc >= 0) {
        const int p = p_acc, e = e0 + p;
        const double* xcol = wd.xcol + (long)w * nsp;
        const double* arow = wd.AinvT[spin] + ((long)w * nsp + p) * nsp;
        double a4[4] = {0, 0, 0, 0};
        for (int j = tid; j < n2; j += PT) {
            const double2 xj = ld2<COH>(xcol + 2 * j);
            const double2 v0 = ld2<COH>(v + 2 * j), v1 = ld2<COH>(v + wd.ldv + 2 * j), v2 = ld2<COH>(v + 2 * wd.ldv + 2 * j), v3 = ld2<COH>(v + 3 * wd.ldv + 2 * j);
            reinterpret_cast<double2*>(vs)[j] = v0;
            reinterpret_cast<double2*>(as)[j] = ldg2(arow + 2 * j);
            a4[0] += v0.x * xj.x + v0.y * xj.y;
            a4[1] += v1.x * xj.x + v1.y * xj.y;
            a4[2] += v2.x * xj.x + v2.y * xj.y;
            a4[3] += v3.x * xj.x + v3.y * xj.y;
        }
        group_sum<PT, 4>(a4, red, tid, sync);
        rho = a4[0];
        if (tid == 0) {
            const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
            const double qx = wd.rp[3 * w], qy = wd.rp[3 * w + 1], qz = wd.rp[3 * w + 2];
            const double Gx = wd.G[3 * w], Gy = wd.G[3 * w + 1], Gz = wd.G[3 * w + 2];
            const double u = wd.u[w], dJ = wd.dJ[w];
            unsigned bits = 0;
            double pacc = 0.0, jr = 0.0;
            bool accept = false;
            if (fabs(rho) < 1e-12) bits |= 2u;
            if (rho > 0.0) {  // fixed node: reject rho_D <= 0 (A7); NaN fails the comparison and rejects
                double Hx = a4[1] / rho + wd.gJn[3 * w], Hy = a4[2] / rho + wd.gJn[3 * w + 1], Hz = a4[3] / rho + wd.gJn[3 * w + 2];
                limit_drift(Hx, Hy, Hz, wd.lim_a, tau);
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
                const double rr = wd.dr2p[w];  // |sqrt(tau) chi|^2 of this proposal (for tau_eff, row f1)
                wd.dr2[2 * w + 1] += rr;
                if (accept) {
                    wd.dr2[2 * w] += rr;
                    Rw[e] = qx; Rw[nep + e] = qy; Rw[2 * nep + e] = qz;
                    wd.logpsi[w] += log(rho) + dJ;
                }
            }
            bc[0] = (accept && commit) ? 1.0 : 0.0;
        }
    }
    sync();  // xs, vs, as, bc[0] and the new position are visible to the block
    if (p_acc >= 0) accepted = bc[0] != 0.0;
    if (!accepted && p_prop < 0) return;

    // ---- one pass over the window rows of earlier kernels: r_l = v . Wbuf[l] (commit), b_l = Vbuf[l] . a_p (proposal)
    if (accepted) {
        double* orb = wd.Orb[spin] + ((long)w * nsp + p_acc) * 5 * nsp;
        for (int j = tid; j < n2; j += PT) {  // row caches and the new window rows: fire-and-forget stores
            const double2 v1 = ld2<COH>(v + wd.ldv + 2 * j), v2 = ld2<COH>(v + 2 * wd.ldv + 2 * j), v3 = ld2<COH>(v + 3 * wd.ldv + 2 * j), v4 = ld2<COH>(v + 4 * wd.ldv + 2 * j);
            const double2 v0 = reinterpret_cast<double2*>(vs)[j];
            reinterpret_cast<double2*>(orb)[j] = v0;
            reinterpret_cast<double2*>(orb + nsp)[j] = v1;
            reinterpret_cast<double2*>(orb + 2 * nsp)[j] = v2;
            reinterpret_cast<double2*>(orb + 3 * nsp)[j] = v3;
            reinterpret_cast<double2*>(orb + 4 * nsp)[j] = v4;
            reinterpret_cast<double2*>(Vb + (long)m_old * nsp)[j] = v0;
            reinterpret_cast<double2*>(Wb + (long)m_old * nsp)[j] = reinterpret_cast<double2*>(as)[j];
        }
        for (int n = tid; n < m_old; n += PT) cs[n] = wd.cvec[(long)w * kp + n];
    }
    if constexpr (PT == 128) {   // short rows (PT = 128 <=> at most 256 orbitals): four rows per warp at a time (same sums, term by term, as the loop below)
        constexpr int R = 4;
        for (int l = warp; l < m_old; l += R * PW) {
            const int nr = (m_old - l + PW - 1) / PW < R ? (m_old - l + PW - 1) / PW : R;
            double ra[R], rb[R];
            const double* rowW = accepted ? Wb + (long)l * nsp : nullptr;
            const double* rowV = p_prop >= 0 ? Vb + (long)l * nsp : nullptr;
            warp_dot2_rows<COH, R>(rowW, vs, rowV, xs, (long)PW * nsp, nr, n2, lane, ra, rb);
            if (lane == 0)
                for (int r = 0; r < nr; r++) {
                    if (accepted) rs[l + r * PW] = ra[r];
                    if (p_prop >= 0) bs[l + r * PW] = rb[r];
                }
        }
    } else
    for (int l = warp; l < m_old; l += PW) {
        double ra = 0.0, rb = 0.0;
        if (accepted && p_prop >= 0) {
            warp_dot2<COH>(Wb + (long)l * nsp, vs, Vb + (long)l * nsp, xs, n2, lane, ra, rb);
            if (lane == 0) { rs[l] = ra; bs[l] = rb; }
        } else if (accepted) {
            warp_dot2<COH>(Wb + (long)l * nsp, vs, nullptr, vs, n2, lane, ra, rb);
            if (lane == 0) rs[l] = ra;
        } else {
            warp_dot2<COH>(Vb + (long)l * nsp, xs, nullptr, xs, n2, lane, ra, rb);
            if (lane == 0) bs[l] = ra;
        }
    }
    if (accepted && p_prop >= 0 && warp == (m_old & (PW - 1))) {  // the row added by this kernel is still in shared memory
        double acc = 0.0;
        for (int j = lane; j < n2; j += 32) {
            const double2 a = reinterpret_cast<double2*>(vs)[j], x = reinterpret_cast<double2*>(xs)[j];
            acc += a.x * x.x + a.y * x.y;
        }
        acc = warp_sum(acc);
        if (lane == 0) bs[m_old] = acc;
    }
    sync();
    if (accepted) {
        // bordered update of S^-1:  t_l = sum_n r_n SinvT[l][n] (one warp per row l)
        const int m = m_old;
        for (int l = warp; l < m; l += PW) {
            double acc = 0.0;
            for (int n = lane; n < m; n += 32) acc += rs[n] * Si[l * kp + n];
            acc = warp_sum(acc);
            if (lane == 0) ts[l] = acc;
        }
        sync();
        const double sinv = 1.0 / rho;
        for (int idx = tid; idx < m * m; idx += PT) {
            const int l = idx / m, n = idx - l * m;
            Si[l * kp + n] += cs[n] * ts[l] * sinv;
        }
        for (int n = tid; n < m; n += PT) {
            Si[m * kp + n] = -cs[n] * sinv;
            Si[n * kp + m] = -ts[n] * sinv;
        }
        if (tid == 0) {
            Si[m * kp + m] = sinv;
            wd.plist[(long)w * kp + m] = p_acc;
            wd.mcount[w] = m + 1;
        }
        sync();  // S^-1 is read again below
    }
    if (p_prop < 0) return;

    // =================================================================== a1 + a2 + a6 for electron p_prop
    const int p = p_prop, e = e0 + p;
    const int m = m_old + (accepted ? 1 : 0);
    if (m > 0) {
        // c = S^-1 b: c_n = sum_l SinvT[l][n] b_l, PT / 128 threads per n over interleaved l, fixed-order combine (kp <= 128)
        constexpr int CP = PT / 128;  // threads per n
        {
            const int n = tid & 127, q = tid >> 7;
            double acc = 0.0;
            if (n < m)
                for (int l = q; l < m; l += CP) acc += Si[l * kp + n] * bs[l];
            c4[q * 128 + n] = acc;
        }
        sync();
        for (int n = tid; n < m; n += PT) {
            const double c = CP == 4 ? (c4[n] + c4[128 + n]) + (c4[256 + n] + c4[384 + n]) : (CP == 2 ? c4[n] + c4[128 + n] : c4[n]);
            cs[n] = c;
            wd.cvec[(long)w * kp + n] = c;
        }
        sync();
        // x = a_p - Wbuf^T c  (effective column of the delayed inverse)
        for (int j = tid; j < n2; j += PT) {
            double2 acc = reinterpret_cast<double2*>(xs)[j];
            int l = 0;
            if constexpr (PT == 128)
            for (; l + 8 <= m_old; l += 8) {
                double2 wv[8];
#pragma unroll
                for (int u = 0; u < 8; u++) wv[u] = ld2<COH>(Wb + (long)(l + u) * nsp + 2 * j);
#pragma unroll
                for (int u = 0; u < 8; u++) { acc.x -= cs[l + u] * wv[u].x; acc.y -= cs[l + u] * wv[u].y; }
            }
            for (; l + 4 <= m_old; l += 4) {
                double2 wv[4];
#pragma unroll
                for (int u = 0; u < 4; u++) wv[u] = ld2<COH>(Wb + (long)(l + u) * nsp + 2 * j);
#pragma unroll
                for (int u = 0; u < 4; u++) { acc.x -= cs[l + u] * wv[u].x; acc.y -= cs[l + u] * wv[u].y; }
            }
            for (; l < m_old; l++) {
                const double2 wv = ld2<COH>(Wb + (long)l * nsp + 2 * j);
                acc.x -= cs[l] * wv.x; acc.y -= cs[l] * wv.y;
            }
            if (accepted) {
                const double2 wv = reinterpret_cast<double2*>(as)[j];
                acc.x -= cs[m_old] * wv.x; acc.y -= cs[m_old] * wv.y;
            }
            reinterpret_cast<double2*>(xs)[j] = acc;
        }
        // each thread reads back only its own xs entries below: no barrier needed
    }
    double* xcol = wd.xcol + (long)w * nsp;
    const double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
    double acc6[6] = {0, 0, 0, 0, 0, 0};
    for (int j = tid; j < n2; j += PT) {
        const double2 xj = reinterpret_cast<double2*>(xs)[j];
        reinterpret_cast<double2*>(xcol)[j] = xj;
        const double2 o1 = ldg2(orb + nsp + 2 * j), o2 = ldg2(orb + 2 * nsp + 2 * j), o3 = ldg2(orb + 3 * nsp + 2 * j);
        acc6[0] += o1.x * xj.x + o1.y * xj.y;
        acc6[1] += o2.x * xj.x + o2.y * xj.y;
        acc6[2] += o3.x * xj.x + o3.y * xj.y;
    }
    // Jastrow gradient at r: grad u = u'(r) (r_i - r_k) / r with u' = a / (1 + b r)^2 -- one sqrt, one division per partner
    const int npart = s.ne + s.n_atoms;
    for (int k = tid; k < npart; k += PT) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double q = 1.0 + P.b * r;
            const double wgt = P.a / (q * q * r);
            acc6[3] += wgt * dx;
            acc6[4] += wgt * dy;
            acc6[5] += wgt * dz;
        }
    }
    group_sum<PT, 6>(acc6, red, tid, sync);
    double Gx = acc6[0] + acc6[3], Gy = acc6[1] + acc6[4], Gz = acc6[2] + acc6[5];
    limit_drift(Gx, Gy, Gz, wd.lim_a, tau);
    const double qx = rx + tau * Gx + sqrt_tau * bc[4];
    const double qy = ry + tau * Gy + sqrt_tau * bc[5];
    const double qz = rz + tau * Gz + sqrt_tau * bc[6];
    if (tid == 0) {
        wd.rp[3 * w] = qx; wd.rp[3 * w + 1] = qy; wd.rp[3 * w + 2] = qz;
        wd.G[3 * w] = Gx; wd.G[3 * w + 1] = Gy; wd.G[3 * w + 2] = Gz;
        wd.u[w] = bc[7];
        wd.dr2p[w] = tau * (bc[4] * bc[4] + bc[5] * bc[5] + bc[6] * bc[6]);
    }
    // Jastrow ratio, term by term, and gradient at r'.  With q = 1 + b r:  u(r') - u(r) = a (r' - r) / (q' q)  (the same
    // term, written without the cancellation of two nearly equal quotients) and grad' = a / (q'^2 r') (r' - r_k);
    // one division t = 1 / (q'^2 q r') serves both: 1/(q' q) = t q' r',  1/(q'^2 r') = t q.
    double acc4[4] = {0, 0, 0, 0};
    for (int k = tid; k < npart; k += PT) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double ex = qx - P.x, ey = qy - P.y, ez = qz - P.z;
            const double r_old = sqrt(dx * dx + dy * dy + dz * dz);
            const double r_new = sqrt(ex * ex + ey * ey + ez * ez);
            const double qo = 1.0 + P.b * r_old, qn = 1.0 + P.b * r_new;
            const double t = P.a / (qn * qn * qo * r_new);
            acc4[0] += (r_new - r_old) * (t * qn * r_new);
            const double wgt = t * qo;
            acc4[1] += wgt * ex;
            acc4[2] += wgt * ey;
            acc4[3] += wgt * ez;
        }
    }
    group_sum<PT, 4>(acc4, red, tid, sync);
    if (tid == 0) {
        wd.dJ[w] = acc4[0];
        wd.gJn[3 * w] = acc4[1]; wd.gJn[3 * w + 1] = acc4[2]; wd.gJn[3 * w + 2] = acc4[3];
    }
}

// p_acc >= 0: finish the move of electron p_acc of this spin (needs its MO rows in V);  p_prop >= 0: propose the
// move of electron p_prop.  commit == 0 evaluates the decision but changes no state (stage timing only).
template <int PT>
__global__ void __launch_bounds__(PT, 1024 / PT) k_step(SysDev s, WalkDev wd, int spin, int p_acc, int p_prop, long log_off, uint32_t step,
                                                double tau, double sqrt_tau, int commit) {
    extern __shared__ __align__(16) double sm[];
    step_body<PT, false>(s, wd, blockIdx.x, threadIdx.x, sm, CtaSync{}, spin, p_acc, p_prop, log_off, step, tau, sqrt_tau, commit);
}

}  // namespace qmc
