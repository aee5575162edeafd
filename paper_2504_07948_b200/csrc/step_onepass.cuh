// step_onepass.cuh -- the per-walker part of one electron step for LARGE systems (rows of the inverse longer than 256):
// rows a5 + a7 of electron p fused with rows a1 + a2 + a6 of electron q = p + 1, as step_kernel.cuh, but with the delay
// window read ONCE.                                                           [BASELINE.json north_star items 3, 4]
//
// step_kernel.cuh forms the effective column of the delayed inverse explicitly, x = a_q - Wbuf^T c, which costs a second
// pass over Wbuf, a round trip of x through HBM, and a chain of phases each exposing a memory latency; its two Jastrow
// passes (2 (N_e + N_a) square roots and divisions per walker) run with the memory system idle.  Here x is never formed.
// Everything the step needs from the window is a dot product of a window row with one of eight vectors:
//     rho_D      = v_0 . x_p   = v_0 . a_p - sum_l c_l (Wbuf_l . v_0)          (v_0: orbital values at r'; c = S^-1 b of p)
//     grad rho_D = v_k . x_p   = v_k . a_p - sum_l c_l (Wbuf_l . v_k)          k = 1..3
//     r_l        = Wbuf_l . v_0                                                 (bordered update of S^-1 on accept)
//     drift of q = o_k . x_q   = o_k . a_q - sum_l c'_l (Wbuf_l . o_k)          (o_k: gradient rows of the row cache of q)
//     b_l        = Vbuf_l . a_q                                                 (c' = S'^-1 b)
// so the kernel is ONE pass in which every load is independent of every other -- the vectors into shared memory, then all
// pending window rows against them -- followed by a short tail on O(m^2) data.  The pass is a skinny GEMM, [8 vectors] x
// [N_s] x [2 m rows]: FP64 DMMA m8n8k4 with the vectors as the A operand (shared memory, conflict-free by the row stride)
// and eight window rows as the B operand, loaded straight from HBM in fragment order (four lanes cover 64 contiguous
// bytes of a row).  The Jastrow sums -- the ratio and gradient at r'_p of the move being decided, the gradient at r_q for
// the drift of the next one -- depend on positions only: they come first, all partner coordinates of a thread requested
// at once (twelve partners per thread in flight), while the rows of the vectors are prefetched into L2.  Bytes per
// walker: 10 rows + 2 m rows + 7 rows stored on accept = SURVEY 8(d).3's count for a1 + a5 + a6 + a7.
//
// State between launches: c of the pending proposal (cvec), its position r', drift G, uniform u.  (The two-pass kernel
// also keeps x, dJ and grad J(r'); this one recomputes the Jastrow terms of the pending proposal in the launch that
// decides it: the positions have not changed in between.)
#pragma once
#include "mo_streamk.cuh"   // dmma884
#include "step_kernel.cuh"

namespace qmc {

// threads per walker: 256, two CTAs to an SM, where the eight vectors of two walkers fit in an SM's shared memory; 512 (one
// CTA to an SM, twice the loads in flight) for longer rows
constexpr int S1_PT_SMALL = 256, S1_PT_LARGE = 512;
constexpr int S1_NX = 8;              // vectors in shared memory, the A operand of the pass: v0 v1 v2 v3 | o1 o2 o3 | a_q
constexpr int S1_ND = 11;             // dot products that need no window row
constexpr int S1_NJ = 7;              // Jastrow sums: grad J at r_q (3) | dJ and grad J at r'_p (4)

struct Step1Layout {
    int ld, vec, part, rw_ld, rw, bs, cs, cn, ts, red, jred, wb, bc, total;   // offsets in doubles
    __host__ __device__ Step1Layout(int nsp, int kp, int S1_PW) {
        ld = nsp + 8;                 // vector stride = 64 B mod 128 B: conflict-free 16-byte fragment loads (see the pass)
        vec = 0;
        part = vec + S1_NX * ld;
        const int ngmax = 2 * ((kp + 7) / 8);
        int psz = S1_PW * ((ngmax + S1_PW - 1) / S1_PW + 1) * 64;   // partial 8 x 8 tiles of the pass; later S1_PW partial column sums of S^-1
        if (psz < S1_PW * kp) psz = S1_PW * kp;
        rw_ld = kp + 1;
        rw = part + psz;
        bs = rw + 7 * rw_ld;
        cs = bs + rw_ld; cn = cs + rw_ld; ts = cn + rw_ld;
        red = ts + rw_ld;
        jred = red + S1_ND * S1_PW;
        wb = jred + S1_NJ * S1_PW;    // 2 (S1_PW + 1) ints: first unit and first group of every warp's range
        bc = wb + S1_PW + 2;
        total = bc + 16;
    }
};
inline size_t step1_smem_bytes(int nsp, int kp, int pt) { return (size_t)Step1Layout(nsp, kp, pt / 32).total * sizeof(double); }
inline int step1_threads(int nsp, int kp) { return 2 * (step1_smem_bytes(nsp, kp, S1_PT_SMALL) + 1024) <= 227 * 1024 ? S1_PT_SMALL : S1_PT_LARGE; }
// the one-pass kernel keeps eight vectors in shared memory
inline bool step1_fits(int nsp, int kp, bool forced) {
    return (nsp > 256 || forced) && step1_smem_bytes(nsp, kp, step1_threads(nsp, kp)) <= 220 * 1024;
}

// 1 / sqrt(x) and 1 / x for the Jastrow sums, branch-free: an FP32 seed (MUFU, 2^-22) and two Newton steps in FP64 (error
// 2^-44, then below the rounding of the steps themselves: about 1 ulp).  The library routines carry a slow path behind a
// branch for arguments outside the FP32 exponent range -- never met here: squared distances in bohr^2 and (1 + b r)^3 --
// and that branch keeps the compiler from interleaving the chains of the partners a thread works on (measured: the sums
// of a launch 11 us with the library calls, each thread 11 partners one after the other).
__device__ __forceinline__ double s1_rsqrt(double x) {
    float y0;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"((float)x));
    double y = (double)y0;
    const double h = 0.5 * x;
    y = y * fma(-(h * y), y, 1.5);
    y = y * fma(-(h * y), y, 1.5);
    return y;
}
__device__ __forceinline__ double s1_rcp(double x) {
    float y0;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"((float)x));
    double y = (double)y0;
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    return y;
}

template <int N>
__device__ __forceinline__ double s1_sum(const double* p) {   // fixed order: pairwise
    if constexpr (N == 1) return p[0];
    else return s1_sum<N / 2>(p) + s1_sum<N / 2>(p + N / 2);
}

// The body works on walker w with the S1_PT threads tid = 0 .. S1_PT - 1 that `sync` joins, in their shared memory `sm`
// (Step1Layout(nsp, kp, S1_PT / 32).total doubles): a whole CTA (k_step1p) or a 128-thread group of the window kernel of the
// mid-size path.  COH: V and the window rows may have been written earlier in the SAME launch (window kernel): they are
// read through L2 (ld.global.cg), not through the non-coherent read-only path.  Every branch that leaves the body is uniform
// over those threads.
template <int S1_PT, bool COH, class Sync>
__device__ __forceinline__ void step1_body(const SysDev& s, const WalkDev& wd, const int w, const int tid, double* sm, const Sync& sync, int spin,
                                           int p_acc, int p_prop, long log_off, uint32_t step, double tau, double sqrt_tau, int commit) {
    constexpr int S1_PW = S1_PT / 32;
    const int lane = tid & 31, warp = tid >> 5;
    const int nsp = s.nsp[spin], n2 = nsp >> 1, kp = wd.kp, nep = wd.nep;
    const int e0 = spin == 0 ? 0 : s.ns[0];
    const Step1Layout L(nsp, kp, S1_PW);
    const int ld = L.ld, rld = L.rw_ld;
    double *vec = sm + L.vec, *part = sm + L.part, *rw = sm + L.rw, *bs = sm + L.bs, *cs = sm + L.cs, *cn = sm + L.cn, *ts = sm + L.ts;
    double *red = sm + L.red, *jred = sm + L.jred, *bc = sm + L.bc;
    int* wbeg = reinterpret_cast<int*>(sm + L.wb);   // [S1_PW + 1] first unit of warp q's range; [S1_PW + 1 ..] its first group
    double* Rw = wd.R + (long)w * 3 * nep;
    double* Vb = wd.Vbuf + (long)w * kp * nsp;
    double* Wb = wd.Wbuf + (long)w * kp * nsp;
    double* Si = wd.SinvT + (long)w * kp * kp;
    const int m_old = wd.mcount[w];
    const bool has_acc = p_acc >= 0, has_prop = p_prop >= 0;
    const int e_acc = e0 + p_acc, e_prop = e0 + p_prop;

    if (has_prop && warp == 1 && lane < 3) {
        // the random numbers of the proposal depend on nothing: one Philox block per lane (reading A11)
        const uint32_t wid = wd.first_walker + (uint32_t)w;
        const uint32_t k0 = (uint32_t)(wd.seed & 0xFFFFFFFFull), k1 = (uint32_t)(wd.seed >> 32);
        uint32_t o[4];
        philox4x32_10(wid, step, (uint32_t)e_prop, (uint32_t)lane, k0, k1, o);
        const double Ua = u01(o[0], o[1]), Ub = u01(o[2], o[3]);
        const double TWO_PI = 6.283185307179586;
        if (lane == 0) { const double r1 = sqrt(-2.0 * log(Ua)); bc[4] = r1 * cos(TWO_PI * Ub); bc[5] = r1 * sin(TWO_PI * Ub); }
        if (lane == 1) { const double r2 = sqrt(-2.0 * log(Ua)); bc[6] = r2 * cos(TWO_PI * Ub); }
        if (lane == 2) bc[7] = Ua;
    }
    // the old S^-1 is read after the pass: have it in L2 by then
    for (int l = tid; l < m_old; l += S1_PT)
        for (int n = 0; n < m_old; n += 16) asm volatile("prefetch.global.L2 [%0];" ::"l"(Si + l * kp + n));
    const double* v = wd.V + (long)w * 5 * wd.ldv;
    const double* arow_p = wd.AinvT[spin] + ((long)w * nsp + (has_acc ? p_acc : 0)) * nsp;
    const double* arow_q = wd.AinvT[spin] + ((long)w * nsp + (has_prop ? p_prop : 0)) * nsp;
    const double* orbq = wd.Orb[spin] + ((long)w * nsp + (has_prop ? p_prop : 0)) * 5 * nsp;
    // ================================================================ the Jastrow sums (reading A5), while the rows below come up from HBM
    // With q = 1 + b r:  grad u = a / (q^2 r) (r_i - r_k);  u(r') - u(r) = a (r' - r) / (q' q), term by term (reading "new").
    // r = d^2 rsqrt(d^2), and ONE reciprocal t = 1 / (q'^2 q) serves the ratio and the gradient at r': 1 / (q' q) = t q',
    // 1 / (q'^2 r') = t q / r'.  All loads of a round of twelve partners per thread first, then their chains.
    {
        const int nline = nsp >> 4;   // 128-byte lines of a row
        for (int i = tid; i < 9 * nline; i += S1_PT) {
            const int r = i / nline, c = (i - r * nline) << 4;
            const double* row = r < 4 ? (has_acc ? v + (long)r * wd.ldv : nullptr)
                              : r == 4 ? (has_acc ? arow_p : nullptr)
                              : r == 5 ? (has_prop ? arow_q : nullptr)
                                       : (has_prop ? orbq + (long)(r - 5) * nsp : nullptr);
            if (row) asm volatile("prefetch.global.L2 [%0];" ::"l"(row + c));
        }
    }
    // what the decision reads from HBM (the pending proposal's drift, uniform and displacement): requested now, parked in
    // shared memory once the Jastrow sums are done
    double dec_scalar = 0.0;
    if (has_acc && tid < 8)
        dec_scalar = tid < 3 ? wd.G[3 * w + tid] : tid == 3 ? wd.u[w] : tid == 4 ? wd.dr2p[w] : tid < 7 ? wd.dr2[2 * w + (tid - 5)] : wd.logpsi[w];
    const int npart = s.ne + s.n_atoms;
    double rx = 0.0, ry = 0.0, rz = 0.0;      // r_q
    double ox = 0.0, oy = 0.0, oz = 0.0;      // r_p
    double px = 0.0, py = 0.0, pz = 0.0;      // r'_p
    if (has_prop) { rx = Rw[e_prop]; ry = Rw[nep + e_prop]; rz = Rw[2 * nep + e_prop]; }
    if (has_acc) {
        ox = Rw[e_acc]; oy = Rw[nep + e_acc]; oz = Rw[2 * nep + e_acc];
        px = wd.rp[3 * w]; py = wd.rp[3 * w + 1]; pz = wd.rp[3 * w + 2];
    }
    auto jastrow_sums = [&]() {
        double jg[S1_NJ];
#pragma unroll
        for (int i = 0; i < S1_NJ; i++) jg[i] = 0.0;
        const bool same_up = e0 == 0;   // (both electrons of a launch are in the same spin block)
        constexpr int JU = 12;
        for (int k0 = tid; k0 < npart; k0 += JU * S1_PT) {
            double kx[JU], ky[JU], kz[JU];
#pragma unroll
            for (int i = 0; i < JU; i++) {   // all loads of the round first
                const int k = k0 + i * S1_PT;
                kx[i] = ky[i] = kz[i] = 0.0;
                if (k < s.ne) {
                    kx[i] = Rw[k]; ky[i] = Rw[nep + k]; kz[i] = Rw[2 * nep + k];
                } else if (k < npart) {
                    const int I = k - s.ne;
                    kx[i] = __ldg(s.atom_xyz + 3 * I); ky[i] = __ldg(s.atom_xyz + 3 * I + 1); kz[i] = __ldg(s.atom_xyz + 3 * I + 2);
                }
            }
#pragma unroll
            for (int i = 0; i < JU; i++) {
                const int k = k0 + i * S1_PT;
                if (k >= npart) continue;
                const bool el = k < s.ne;
                const double a = el ? (((k < s.ns[0]) == same_up) ? s.a_para : s.a_anti) : -__ldg(s.atom_Z + (k - s.ne));
                const double b = el ? s.b_ee : s.b_en;
                if (has_prop && k != e_prop && !(has_acc && k == e_acc)) {   // (electron e_acc may still move: its term follows the decision)
                    const double dx = rx - kx[i], dy = ry - ky[i], dz = rz - kz[i];
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    const double ir = s1_rsqrt(d2);
                    const double q = 1.0 + b * (d2 * ir);
                    const double wgt = a * ir * s1_rcp(q * q);
                    jg[0] += wgt * dx; jg[1] += wgt * dy; jg[2] += wgt * dz;
                }
                if (has_acc && k != e_acc) {
                    const double dx = ox - kx[i], dy = oy - ky[i], dz = oz - kz[i];
                    const double ex = px - kx[i], ey = py - ky[i], ez = pz - kz[i];
                    const double d2o = dx * dx + dy * dy + dz * dz, d2n = ex * ex + ey * ey + ez * ez;
                    const double iro = s1_rsqrt(d2o), irn = s1_rsqrt(d2n);
                    const double r_old = d2o > 0.0 ? d2o * iro : 0.0, r_new = d2n > 0.0 ? d2n * irn : 0.0;
                    const double qo = 1.0 + b * r_old, qn = 1.0 + b * r_new;
                    const double t = a * s1_rcp(qn * qn * qo);
                    jg[3] += (r_new - r_old) * (t * qn);
                    const double wgt = t * qo * irn;
                    jg[4] += wgt * ex; jg[5] += wgt * ey; jg[6] += wgt * ez;
                }
            }
        }
#pragma unroll
        for (int i = 0; i < S1_NJ; i++) {
            const double t = warp_sum(jg[i]);
            if (lane == 0) jred[i * S1_PW + warp] = t;
        }
    };
    jastrow_sums();

    // ================================================================ the vectors, and every dot product that needs no window row
    {
        // acc: 0..3 v_k . a_p | 4..6 o_k . a_q | 7 v_0 . a_q | 8..10 a_p . o_k
        double acc[S1_ND];
#pragma unroll
        for (int i = 0; i < S1_ND; i++) acc[i] = 0.0;
        const int h = ld >> 1;
        for (int j = tid; j < n2; j += S1_PT) {
            const double2 z = make_double2(0.0, 0.0);
            double2 v0 = z, v1 = z, v2 = z, v3 = z, ap = z, aq = z, o1 = z, o2 = z, o3 = z;
            if (has_acc) {
                v0 = ld2<COH>(v + 2 * j); v1 = ld2<COH>(v + wd.ldv + 2 * j); v2 = ld2<COH>(v + 2 * wd.ldv + 2 * j); v3 = ld2<COH>(v + 3 * wd.ldv + 2 * j);
                ap = ldg2(arow_p + 2 * j);
            }
            if (has_prop) {
                aq = ldg2(arow_q + 2 * j);
                o1 = ldg2(orbq + nsp + 2 * j); o2 = ldg2(orbq + 2 * nsp + 2 * j); o3 = ldg2(orbq + 3 * nsp + 2 * j);
            }
            double2* dst = reinterpret_cast<double2*>(vec) + j;
            dst[0] = v0; dst[h] = v1; dst[2 * h] = v2; dst[3 * h] = v3;
            dst[4 * h] = o1; dst[5 * h] = o2; dst[6 * h] = o3; dst[7 * h] = aq;
            acc[0] += v0.x * ap.x + v0.y * ap.y;
            acc[1] += v1.x * ap.x + v1.y * ap.y;
            acc[2] += v2.x * ap.x + v2.y * ap.y;
            acc[3] += v3.x * ap.x + v3.y * ap.y;
            acc[4] += o1.x * aq.x + o1.y * aq.y;
            acc[5] += o2.x * aq.x + o2.y * aq.y;
            acc[6] += o3.x * aq.x + o3.y * aq.y;
            acc[7] += v0.x * aq.x + v0.y * aq.y;
            acc[8] += ap.x * o1.x + ap.y * o1.y;
            acc[9] += ap.x * o2.x + ap.y * o2.y;
            acc[10] += ap.x * o3.x + ap.y * o3.y;
        }
#pragma unroll
        for (int i = 0; i < S1_ND; i++) {
            const double t = warp_sum(acc[i]);
            if (lane == 0) red[i * S1_PW + warp] = t;
        }
    }
    if (has_acc)
        for (int n = tid; n < m_old; n += S1_PT) cs[n] = wd.cvec[(long)w * kp + n];
    // Work units of the pass are (group of eight window rows, step of 16 orbitals), Wbuf groups first, then Vbuf groups; the
    // flattened space is cut into S1_PW equal contiguous ranges, one per warp (stream-K in miniature: every warp streams the
    // same number of bytes whatever m is).  A range crosses at most MAXSEG groups; each crossing leaves one partial tile.
    const int G = (m_old + 7) >> 3;              // groups of eight window rows
    const int NG = has_prop ? 2 * G : G;
    const int St = nsp >> 4;                     // steps per group
    const int U = NG * St;
    const int MAXSEG = (NG + S1_PW - 1) / S1_PW + 1;
    if (tid <= S1_PW) {
        const int b = (int)((long)tid * U / S1_PW);
        wbeg[tid] = b;
        wbeg[S1_PW + 1 + tid] = b / St;
    }
    sync();   // vec, red, cs, wbeg, bc[4..7]

    // ================================================================ the pass over the window: [8 vectors] x [N_s] x [8 rows] DMMA tiles
    if (m_old > 0) {
        const int lr = lane >> 2, lc = lane & 3;
        const int a0 = wbeg[warp], a1 = wbeg[warp + 1];
        constexpr int UN = 8;                    // steps per batch: 16 independent 16-byte loads in flight per lane
        // lane (lr, lc) owns orbitals 16 st + 2 lc + {0, 1} and 16 st + 8 + 2 lc + {0, 1} of window row lr (B operand) and of
        // vector lr (A operand): k index lc of four DMMAs per step
        const double* av = vec + lr * ld + 2 * lc;
        int seg = 0, gg = wbeg[S1_PW + 1 + warp];
        for (int u = a0; u < a1; seg++, gg++) {
            const int s0 = u - gg * St;
            const int s1 = St - s0 < a1 - u ? St : s0 + (a1 - u);
            const bool isV = gg >= G;
            int row = 8 * (isV ? gg - G : gg) + lr;
            if (row >= m_old) row = m_old - 1;   // (a group's missing rows: any valid row, the result is dropped)
            const double* src = (isV ? Vb : Wb) + (long)row * nsp + 2 * lc;
            double d[4][2];
#pragma unroll
            for (int i = 0; i < 4; i++) d[i][0] = d[i][1] = 0.0;
            for (int st = s0; st < s1; st += UN) {
                double2 b[UN][2];
#pragma unroll
                for (int q = 0; q < UN; q++) {
                    const bool on = st + q < s1;   // (past the range: zeros -- the DMMAs add nothing)
                    b[q][0] = on ? ld2<COH>(src + 16 * (st + q)) : make_double2(0.0, 0.0);
                    b[q][1] = on ? ld2<COH>(src + 16 * (st + q) + 8) : make_double2(0.0, 0.0);
                }
#pragma unroll
                for (int q = 0; q < UN; q++) {
                    const int sq = st + q < St ? st + q : St - 1;
                    const double2 x0 = *reinterpret_cast<const double2*>(av + 16 * sq);
                    const double2 x1 = *reinterpret_cast<const double2*>(av + 16 * sq + 8);
                    dmma884(d[0][0], d[0][1], x0.x, b[q][0].x);
                    dmma884(d[1][0], d[1][1], x0.y, b[q][0].y);
                    dmma884(d[2][0], d[2][1], x1.x, b[q][1].x);
                    dmma884(d[3][0], d[3][1], x1.y, b[q][1].y);
                }
            }
            // D[vector lr][row 2 lc + {0, 1}]
            *reinterpret_cast<double2*>(part + (warp * MAXSEG + seg) * 64 + lr * 8 + 2 * lc) =
                make_double2((d[0][0] + d[1][0]) + (d[2][0] + d[3][0]), (d[0][1] + d[1][1]) + (d[2][1] + d[3][1]));
            u += s1 - s0;
        }
    }
    if (tid < 8) bc[8 + tid] = dec_scalar;
    sync();
    // partial tiles summed in ascending order of the orbital index: rw[i][l] = Wbuf_l . (vector i), i = 0..6;  bs[l] = Vbuf_l . a_q
    for (int idx = tid; idx < m_old * 8; idx += S1_PT) {
        const int l = idx >> 3, i = idx & 7, n = l & 7;
        if (i == 7 && !has_prop) continue;
        const int gg = (i < 7 ? 0 : G) + (l >> 3);
        const int u0 = gg * St, u1 = u0 + St;
        double sacc = 0.0;
#pragma unroll
        for (int q = 0; q < S1_PW; q++) {
            const int b0 = wbeg[q], b1 = wbeg[q + 1];
            if (b1 > u0 && b0 < u1 && b1 > b0) sacc += part[(q * MAXSEG + (gg - wbeg[S1_PW + 1 + q])) * 64 + i * 8 + n];
        }
        if (i < 7) rw[i * rld + l] = sacc; else bs[l] = sacc;
    }
    sync();

    // ================================================================ a5 + a7: the decision for electron p_acc
    bool accepted = false;
    double rho = 1.0;
    if (has_acc) {
        unsigned bits = 0;
        double pacc = 0.0, jr = 0.0, dJ = 0.0;
        if (warp == 0) {
            double a4[4] = {0.0, 0.0, 0.0, 0.0};
            for (int l = lane; l < m_old; l += 32) {
                const double c = cs[l];
#pragma unroll
                for (int k = 0; k < 4; k++) a4[k] += c * rw[k * rld + l];
            }
#pragma unroll
            for (int k = 0; k < 4; k++) a4[k] = s1_sum<S1_PW>(red + k * S1_PW) - warp_sum(a4[k]);
            if (lane == 0) {
                rho = a4[0];
                const double Gx = bc[8], Gy = bc[9], Gz = bc[10], u = bc[11];
                dJ = s1_sum<S1_PW>(jred + 3 * S1_PW);
                const double gJx = s1_sum<S1_PW>(jred + 4 * S1_PW), gJy = s1_sum<S1_PW>(jred + 5 * S1_PW), gJz = s1_sum<S1_PW>(jred + 6 * S1_PW);
                bool accept = false;
                if (fabs(rho) < 1e-12) bits |= 2u;
                if (rho > 0.0) {  // fixed node: reject rho_D <= 0 (A7); NaN fails the comparison and rejects
                    double Hx = a4[1] / rho + gJx, Hy = a4[2] / rho + gJy, Hz = a4[3] / rho + gJz;
                    limit_drift(Hx, Hy, Hz, wd.lim_a, tau);
                    const double ax = px - ox - tau * Gx, ay = py - oy - tau * Gy, az = pz - oz - tau * Gz;
                    const double cx = ox - px - tau * Hx, cy = oy - py - tau * Hy, cz = oz - pz - tau * Hz;
                    const double fwd = ax * ax + ay * ay + az * az, rev = cx * cx + cy * cy + cz * cz;
                    const double Delta = (fwd - rev) / (2.0 * tau);
                    pacc = rho * rho * exp(2.0 * dJ + Delta);  // A25: linear domain, one exp
                    if (fabs(u - pacc) < 1e-12) bits |= 2u;
                    accept = (u < pacc);
                }
                if (isnan(rho) || isnan(pacc)) { bits |= 4u; accept = false; }
                if (accept) bits |= 1u;
                bc[0] = (accept && commit) ? 1.0 : 0.0;
                bc[1] = rho;
            }
        }
        sync();  // bc[0], bc[1]
        accepted = bc[0] != 0.0;
        if (tid == 0 && commit) {   // the record of the decision: nobody in this launch waits for it
            if (rho > 0.0) jr = rho * exp(dJ);
            wd.bits[log_off + w] = (uint8_t)bits;
            if (wd.ratio_log) { wd.ratio_log[log_off + w] = jr; wd.pacc_log[log_off + w] = pacc; }
            atomicAdd(&wd.stats[0], 1ull);
            if (accepted) atomicAdd(&wd.stats[1], 1ull);
            if (bits & 2u) atomicAdd(&wd.stats[2], 1ull);
            if (bits & 4u) { atomicAdd(&wd.stats[3], 1ull); wd.flags[w] = 1u; }
            const double rr = bc[12];   // |sqrt(tau) chi|^2 of this proposal (for tau_eff, row f1)
            wd.dr2[2 * w + 1] = bc[14] + rr;
            if (accepted) {
                wd.dr2[2 * w] = bc[13] + rr;
                Rw[e_acc] = px; Rw[nep + e_acc] = py; Rw[2 * nep + e_acc] = pz;
                wd.logpsi[w] = bc[15] + (log(rho) + dJ);
            }
        }
        rho = bc[1];
    }
    if (!accepted && !has_prop) return;
    const double sinv = 1.0 / rho;
    const int m = m_old;
    // the two rows of the commit that are not in shared memory (Laplacian row, a_p): requested now, stored at the end
    constexpr int SR = 2;
    double2 v4r[SR], apr[SR];
#pragma unroll
    for (int i = 0; i < SR; i++) {
        const int j = tid + i * S1_PT;
        v4r[i] = apr[i] = make_double2(0.0, 0.0);
        if (accepted && j < n2) { v4r[i] = ld2<COH>(v + 4 * wd.ldv + 2 * j); apr[i] = ldg2(arow_p + 2 * j); }
    }

    // ---- one pass over the old S^-1: t_l = sum_n r_n SinvT[l][n] (bordered update) and y_n = sum_l SinvT[l][n] b_l (c' = S'^-1 b')
    double* ypart = part;   // [S1_PW][kp]
    if (m > 0) {
        const double* rs = rw;   // r_l = Wbuf_l . v_0
        double y[4] = {0.0, 0.0, 0.0, 0.0};
        const int njj = (m + 31) >> 5;
        for (int l0 = warp; l0 < m; l0 += 4 * S1_PW) {   // four rows per warp at a time, all their loads first
            double sv[4][4];
#pragma unroll
            for (int i = 0; i < 4; i++)
#pragma unroll
                for (int jj = 0; jj < 4; jj++) {
                    const int l = l0 + i * S1_PW, n = lane + 32 * jj;
                    sv[i][jj] = (jj < njj && l < m && n < m) ? Si[l * kp + n] : 0.0;
                }
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const int l = l0 + i * S1_PW;
                if (l >= m) break;
                const double bl = has_prop ? bs[l] : 0.0;
                double tacc = 0.0;
#pragma unroll
                for (int jj = 0; jj < 4; jj++) {
                    const int n = lane + 32 * jj;
                    if (n < m) { tacc += rs[n] * sv[i][jj]; y[jj] += sv[i][jj] * bl; }
                }
                tacc = warp_sum(tacc);
                if (lane == 0) ts[l] = tacc;
                if (accepted) {   // the bordered S^-1, row l, from the values just read: SinvT[l][n] += c_n t_l / rho, SinvT[l][m] = -t_l / rho
                    const double tl = tacc * sinv;
#pragma unroll
                    for (int jj = 0; jj < 4; jj++) {
                        const int n = lane + 32 * jj;
                        if (n < m) Si[l * kp + n] = sv[i][jj] + cs[n] * tl;
                    }
                    if (lane == 0) Si[l * kp + m] = -tl;
                }
            }
        }
#pragma unroll
        for (int jj = 0; jj < 4; jj++) {
            const int n = lane + 32 * jj;
            if (n < m) ypart[warp * kp + n] = y[jj];
        }
    }
    sync();
    if (has_prop) {
        // c'_n = y_n + c_n (tb - b_m) / rho (n < m),  c'_m = (b_m - tb) / rho,  tb = sum_l t_l b_l;  without an accepted move c' = y
        double tb = 0.0;
        if (accepted) {
            for (int l = lane; l < m; l += 32) tb += ts[l] * bs[l];
            tb = warp_sum(tb);   // (every warp the same sum in the same order)
        }
        const double bm = s1_sum<S1_PW>(red + 7 * S1_PW);   // Vbuf_m . a_q = v_0 . a_q
        for (int n = tid; n < m; n += S1_PT) {
            double c = 0.0;
#pragma unroll
            for (int q = 0; q < S1_PW; q++) c += ypart[q * kp + n];
            if (accepted) c += cs[n] * (sinv * (tb - bm));
            cn[n] = c;
            wd.cvec[(long)w * kp + n] = c;
        }
        if (accepted && tid == 0) {
            const double c = sinv * (bm - tb);
            cn[m] = c;
            wd.cvec[(long)w * kp + m] = c;
        }
        sync();   // cn

        // ============================================================ a1 + a2 for electron p_prop (a6: the Jastrow sums above)
        if (warp == 0) {
        double e3[3] = {0.0, 0.0, 0.0};
        for (int l = lane; l < m; l += 32) {
            const double c = cn[l];
#pragma unroll
            for (int k = 0; k < 3; k++) e3[k] += c * rw[(4 + k) * rld + l];
        }
#pragma unroll
        for (int k = 0; k < 3; k++) e3[k] = warp_sum(e3[k]);
        const double cm = accepted ? cn[m] : 0.0;
        double Gx = s1_sum<S1_PW>(red + 4 * S1_PW) - e3[0] - cm * s1_sum<S1_PW>(red + 8 * S1_PW) + s1_sum<S1_PW>(jred);
        double Gy = s1_sum<S1_PW>(red + 5 * S1_PW) - e3[1] - cm * s1_sum<S1_PW>(red + 9 * S1_PW) + s1_sum<S1_PW>(jred + S1_PW);
        double Gz = s1_sum<S1_PW>(red + 6 * S1_PW) - e3[2] - cm * s1_sum<S1_PW>(red + 10 * S1_PW) + s1_sum<S1_PW>(jred + 2 * S1_PW);
        if (has_acc && e_acc != e_prop) {   // the partner that may just have moved
            const double kx = accepted ? px : ox, ky = accepted ? py : oy, kz = accepted ? pz : oz;
            const double dx = rx - kx, dy = ry - ky, dz = rz - kz;
            const double d2 = dx * dx + dy * dy + dz * dz;
            const double ir = s1_rsqrt(d2);
            const double q = 1.0 + s.b_ee * (d2 * ir);
            const double wgt = s.a_para * ir * s1_rcp(q * q);
            Gx += wgt * dx; Gy += wgt * dy; Gz += wgt * dz;
        }
        limit_drift(Gx, Gy, Gz, wd.lim_a, tau);
        if (tid == 0) {
            wd.rp[3 * w] = rx + tau * Gx + sqrt_tau * bc[4];
            wd.rp[3 * w + 1] = ry + tau * Gy + sqrt_tau * bc[5];
            wd.rp[3 * w + 2] = rz + tau * Gz + sqrt_tau * bc[6];
            wd.G[3 * w] = Gx; wd.G[3 * w + 1] = Gy; wd.G[3 * w + 2] = Gz;
            wd.u[w] = bc[7];
            wd.dr2p[w] = tau * (bc[4] * bc[4] + bc[5] * bc[5] + bc[6] * bc[6]);
        }
        }
    }
    // ---- the row caches, the new window rows and the bordered S^-1, last: nothing in this launch reads them again
    if (accepted) {
        double* orb = wd.Orb[spin] + ((long)w * nsp + p_acc) * 5 * nsp;
        const int h = ld >> 1;
        int it = 0;
        for (int j = tid; j < n2; j += S1_PT, it++) {
            double2 v4, ap;
            if (it == 0) { v4 = v4r[0]; ap = apr[0]; }
            else if (it == 1) { v4 = v4r[1]; ap = apr[1]; }
            else { v4 = ld2<COH>(v + 4 * wd.ldv + 2 * j); ap = ldg2(arow_p + 2 * j); }   // (longer rows: L2 has them)
            const double2* srcv = reinterpret_cast<const double2*>(vec) + j;
            const double2 v0 = srcv[0];
            reinterpret_cast<double2*>(orb)[j] = v0;
            reinterpret_cast<double2*>(orb + nsp)[j] = srcv[h];
            reinterpret_cast<double2*>(orb + 2 * nsp)[j] = srcv[2 * h];
            reinterpret_cast<double2*>(orb + 3 * nsp)[j] = srcv[3 * h];
            reinterpret_cast<double2*>(orb + 4 * nsp)[j] = v4;
            reinterpret_cast<double2*>(Vb + (long)m * nsp)[j] = v0;
            reinterpret_cast<double2*>(Wb + (long)m * nsp)[j] = ap;
        }
        for (int n = tid; n < m; n += S1_PT) Si[m * kp + n] = -cs[n] * sinv;   // (rows 0 .. m - 1 were rewritten in the pass over S^-1)
        if (tid == 0) {
            Si[m * kp + m] = sinv;
            wd.plist[(long)w * kp + m] = p_acc;
            wd.mcount[w] = m + 1;
        }
    }
}

// p_acc >= 0: finish the move of electron p_acc of this spin (needs its MO rows in V);  p_prop >= 0: propose the move of
// electron p_prop.  commit == 0 evaluates the decision but changes no state (stage timing only).
template <int S1_PT>
__global__ void __launch_bounds__(S1_PT, S1_PT == S1_PT_SMALL ? 2 : 1) k_step1p(SysDev s, WalkDev wd, int spin, int p_acc, int p_prop, long log_off, uint32_t step,
                                                                                double tau, double sqrt_tau, int commit) {
    extern __shared__ __align__(16) double sm[];
    step1_body<S1_PT, false>(s, wd, blockIdx.x, threadIdx.x, sm, CtaSync{}, spin, p_acc, p_prop, log_off, step, tau, sqrt_tau, commit);
}

}  // namespace qmc
