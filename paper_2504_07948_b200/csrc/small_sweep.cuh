// small_sweep.cuh -- row f4 of SURVEY 8(f): the paper's own regime (8-240 electrons, thousands of walkers per GPU,
// PAPER.md L265, L279-302), where the per-electron kernels of the large-system path are pure launch latency (the paper's
// own finding, L157, L265).  For systems with at most 32 electrons per spin whose per-walker state fits in shared
// memory, qmc_sweep / qmc_dmc_step run ALL sweeps of a call in ONE launch: one warp per walker, the walker's
// positions, both A^-1 and the orbital row caches resident in shared memory, the MO coefficients shared by the block.
// Every step is the same arithmetic as the large-system kernels (k_basis, k_mo_streamk, k_step, k_eloc_*), with the
// rank-1 Sherman-Morrison update in place of the delayed one (delay_k only changes rounding, reading A13).
#pragma once
#include "device_utils.cuh"
#include "mo_streamk.cuh"
#include "step_kernel.cuh"

namespace qmc {

struct SmallArgs {
    int nsteps;
    uint32_t step0;
    double tau, sqrt_tau;
    int dmc;          // 1: DMC generation (weights), lim_a in wd.lim_a
    double e_trial;
    const double* e_trial_dev;  // non-null: E_T is read from the device (qmc_dmc_run)
    int nsm;          // max(ns[0], ns[1])
    int wpb;          // warps (walkers) per block
};

__host__ __device__ inline size_t small_block_doubles(const SysDev& s, int nsm) { return (size_t)2 * s.n_basis * nsm; }
__host__ __device__ inline size_t small_walker_doubles(const SysDev& s, int nep, int nsm) {
    return (size_t)3 * nep + 2 * nsm * nsm + 2 * nsm * 5 * nsm + 5 * s.n_basis + 5 * nsm;
}

__global__ void __launch_bounds__(256) k_sweep_small(SysDev s, WalkDev wd, SmallArgs a) {
    extern __shared__ __align__(16) double ssm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nb = s.n_basis, nsm = a.nsm, nep = wd.nep, ne = s.ne;
    double* Cs = ssm;  // [2][nb][nsm]
    for (int idx = threadIdx.x; idx < 2 * nb * nsm; idx += blockDim.x) {
        const int sp = idx / (nb * nsm), rem = idx - sp * nb * nsm, l = rem / nsm, j = rem - l * nsm;
        Cs[idx] = j < s.ns[sp] ? s.CT[sp][cT_index(l, j, s.kb)] : 0.0;
    }
    __syncthreads();
    const int w = blockIdx.x * a.wpb + warp;
    if (w >= wd.W) return;
    double* Rs = ssm + small_block_doubles(s, nsm) + (size_t)warp * small_walker_doubles(s, nep, nsm);
    double* As = Rs + 3 * nep;              // [2][nsm][nsm]   As[sp][q][j] = (A^-1)[j][q]
    double* Os = As + 2 * nsm * nsm;        // [2][nsm][5][nsm]
    double* phi = Os + 2 * nsm * 5 * nsm;   // [5][nb]
    double* vs = phi + 5 * nb;              // [5][nsm]
    // ---- walker state HBM -> shared memory
    for (int i = lane; i < 3 * nep; i += 32) Rs[i] = wd.R[(long)w * 3 * nep + i];
    for (int sp = 0; sp < 2; sp++) {
        const int ns = s.ns[sp], nsp = s.nsp[sp];
        for (int idx = lane; idx < ns * ns; idx += 32) {
            const int q = idx / ns, j = idx - q * ns;
            As[(sp * nsm + q) * nsm + j] = wd.AinvT[sp][((long)w * nsp + q) * nsp + j];
        }
        for (int idx = lane; idx < ns * 5 * ns; idx += 32) {
            const int q = idx / (5 * ns), rem = idx - q * 5 * ns, c = rem / ns, j = rem - c * ns;
            Os[((sp * nsm + q) * 5 + c) * nsm + j] = wd.Orb[sp][(((long)w * nsp + q) * 5 + c) * nsp + j];
        }
    }
    double logpsi = wd.logpsi[w], weight = wd.weight[w], e_old = wd.eloc[w];
    const double e_trial = a.e_trial_dev ? *a.e_trial_dev : a.e_trial;
    unsigned long long n_acc = 0, n_tie = 0, n_nonf = 0;
    const uint32_t wid = wd.first_walker + (uint32_t)w;
    const uint32_t k0 = (uint32_t)(wd.seed & 0xFFFFFFFFull), k1 = (uint32_t)(wd.seed >> 32);
    const int npart = ne + s.n_atoms;
    const double tau = a.tau;
    __syncwarp();

    for (int t = 0; t < a.nsteps; t++) {
        double dr2_acc = 0.0, dr2_all = 0.0;
        for (int e = 0; e < ne; e++) {
            const int sp = e < s.ns[0] ? 0 : 1, p = sp ? e - s.ns[0] : e, ns = s.ns[sp];
            double* A = As + sp * nsm * nsm;
            double* Op = Os + ((sp * nsm + p) * 5) * nsm;
            const double xj = lane < ns ? A[p * nsm + lane] : 0.0;  // row p of A^-T: the column the ratio needs
            // ---- a1: drift
            const double rx = Rs[e], ry = Rs[nep + e], rz = Rs[2 * nep + e];
            double g0 = 0, g1 = 0, g2 = 0;
            if (lane < ns) { g0 = Op[nsm + lane] * xj; g1 = Op[2 * nsm + lane] * xj; g2 = Op[3 * nsm + lane] * xj; }
            double j0 = 0, j1 = 0, j2 = 0;
            for (int k = lane; k < npart; k += 32) {
                Partner P = partner(s, Rs, nep, e, k);
                if (P.ok) {
                    const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
                    const double r = sqrt(dx * dx + dy * dy + dz * dz);
                    const double q = 1.0 + P.b * r;
                    const double wgt = P.a / (q * q * r);
                    j0 += wgt * dx; j1 += wgt * dy; j2 += wgt * dz;
                }
            }
            double Gx = warp_sum(g0) + warp_sum(j0), Gy = warp_sum(g1) + warp_sum(j1), Gz = warp_sum(g2) + warp_sum(j2);
            limit_drift(Gx, Gy, Gz, wd.lim_a, tau);
            // ---- a2: Philox proposal (one block per lane 0..2, reading A11)
            double c0 = 0, c1 = 0;
            if (lane < 3) {
                uint32_t o[4];
                philox4x32_10(wid, a.step0 + (uint32_t)t, (uint32_t)e, (uint32_t)lane, k0, k1, o);
                const double Ua = u01(o[0], o[1]), Ub = u01(o[2], o[3]);
                const double TWO_PI = 6.283185307179586;
                if (lane == 2) c0 = Ua;
                else {
                    const double rr = sqrt(-2.0 * log(Ua));
                    c0 = rr * cos(TWO_PI * Ub);
                    if (lane == 0) c1 = rr * sin(TWO_PI * Ub);
                }
            }
            const double chx = __shfl_sync(0xffffffffu, c0, 0), chy = __shfl_sync(0xffffffffu, c1, 0);
            const double chz = __shfl_sync(0xffffffffu, c0, 1), u = __shfl_sync(0xffffffffu, c0, 2);
            const double rr2 = tau * (chx * chx + chy * chy + chz * chz);
            const double qx = rx + tau * Gx + a.sqrt_tau * chx, qy = ry + tau * Gy + a.sqrt_tau * chy, qz = rz + tau * Gz + a.sqrt_tau * chz;
            // ---- a3: basis functions at r' (a lane per shell)
            for (int sh = lane; sh < s.n_shells; sh += 32) {
                const ShellRec rec = s.shells[sh];
                const double x = qx - rec.x, y = qy - rec.y, z = qz - rec.z;
                const double tt = x * x + y * y + z * z;
                double g = 0.0, gp = 0.0, gpp = 0.0;
                for (int q = 0; q < rec.nprim; q++) {
                    const double al = __ldg(s.alpha + rec.poff + q);
                    const double ee = __ldg(s.coef + rec.poff + q) * exp(-al * tt);
                    g += ee;
                    gp -= al * ee;
                    gpp += al * al * ee;
                }
                const double lapfac = (double)(4 * rec.l + 6) * gp + 4.0 * tt * gpp;
                const double tg1 = 2.0 * gp;
                auto emit = [&](int m, double S, double Sx, double Sy, double Sz) {
                    const int f = rec.f0 + m;
                    phi[f] = S * g;
                    phi[nb + f] = g * Sx + tg1 * S * x;
                    phi[2 * nb + f] = g * Sy + tg1 * S * y;
                    phi[3 * nb + f] = g * Sz + tg1 * S * z;
                    phi[4 * nb + f] = S * lapfac;
                };
                const double s3 = 1.7320508075688772;
                if (rec.l == 0) {
                    emit(0, 1.0, 0.0, 0.0, 0.0);
                } else if (rec.l == 1) {
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
            __syncwarp();
            // ---- a4: MO rows v[c][j] = sum_l C[l][j] phi[c][l]
            const double* C = Cs + (size_t)sp * nb * nsm;
            for (int idx = lane; idx < 5 * ns; idx += 32) {
                const int c = idx / ns, j = idx - c * ns;
                double acc = 0.0;
                for (int l = 0; l < nb; l++) acc += C[l * nsm + j] * phi[c * nb + l];
                vs[c * nsm + j] = acc;
            }
            __syncwarp();
            // ---- a5: determinant ratio and gradient at r'
            double r0 = 0, r1 = 0, r2 = 0, r3 = 0;
            if (lane < ns) { r0 = vs[lane] * xj; r1 = vs[nsm + lane] * xj; r2 = vs[2 * nsm + lane] * xj; r3 = vs[3 * nsm + lane] * xj; }
            const double rho = warp_sum(r0), d1 = warp_sum(r1), d2 = warp_sum(r2), d3 = warp_sum(r3);
            // ---- a6: Jastrow ratio (term by term) and gradient at r'
            double a0 = 0, a1 = 0, a2 = 0, a3 = 0;
            for (int k = lane; k < npart; k += 32) {
                Partner P = partner(s, Rs, nep, e, k);
                if (P.ok) {
                    const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
                    const double ex = qx - P.x, ey = qy - P.y, ez = qz - P.z;
                    const double r_old = sqrt(dx * dx + dy * dy + dz * dz);
                    const double r_new = sqrt(ex * ex + ey * ey + ez * ez);
                    const double qo = 1.0 + P.b * r_old, qn = 1.0 + P.b * r_new;
                    const double tq = P.a / (qn * qn * qo * r_new);
                    a0 += (r_new - r_old) * (tq * qn * r_new);
                    const double wgt = tq * qo;
                    a1 += wgt * ex; a2 += wgt * ey; a3 += wgt * ez;
                }
            }
            const double dJ = warp_sum(a0), gJx = warp_sum(a1), gJy = warp_sum(a2), gJz = warp_sum(a3);
            // ---- a7: accept / reject (every lane holds the same numbers)
            unsigned bits = 0;
            double pacc = 0.0, jr = 0.0;
            bool accept = false;
            if (fabs(rho) < 1e-12) bits |= 2u;
            if (rho > 0.0) {
                double Hx = d1 / rho + gJx, Hy = d2 / rho + gJy, Hz = d3 / rho + gJz;
                limit_drift(Hx, Hy, Hz, wd.lim_a, tau);
                const double ax = qx - rx - tau * Gx, ay = qy - ry - tau * Gy, az = qz - rz - tau * Gz;
                const double cx = rx - qx - tau * Hx, cy = ry - qy - tau * Hy, cz = rz - qz - tau * Hz;
                const double fwd = ax * ax + ay * ay + az * az, rev = cx * cx + cy * cy + cz * cz;
                const double Delta = (fwd - rev) / (2.0 * tau);
                pacc = rho * rho * exp(2.0 * dJ + Delta);
                jr = rho * exp(dJ);
                if (fabs(u - pacc) < 1e-12) bits |= 2u;
                accept = (u < pacc);
            }
            const bool nonfinite = isnan(rho) || isnan(pacc);
            if (nonfinite) { bits |= 4u; accept = false; n_nonf++; }
            if (accept) bits |= 1u;
            if (bits & 2u) n_tie++;
            dr2_all += rr2;
            if (lane == 0) {
                const long lo = ((long)t * ne + e) * wd.W + w;
                wd.bits[lo] = (uint8_t)bits;
                if (wd.ratio_log) { wd.ratio_log[lo] = jr; wd.pacc_log[lo] = pacc; }
            }
            if (accept) {
                n_acc++;
                dr2_acc += rr2;
                logpsi += log(rho) + dJ;
                // Sherman-Morrison on A^-T: row q -= row p * (v . row q) / rho (q != p); row p /= rho
                for (int q = 0; q < ns; q++) {
                    if (q == p) continue;
                    const double aq = lane < ns ? A[q * nsm + lane] : 0.0;
                    const double sq = warp_sum(lane < ns ? vs[lane] * aq : 0.0);
                    if (lane < ns) A[q * nsm + lane] = aq - xj * sq / rho;
                }
                if (lane < ns) A[p * nsm + lane] = xj / rho;
                for (int idx = lane; idx < 5 * ns; idx += 32) {
                    const int c = idx / ns, j = idx - c * ns;
                    Op[c * nsm + j] = vs[c * nsm + j];
                }
                if (lane == 0) { Rs[e] = qx; Rs[nep + e] = qy; Rs[2 * nep + e] = qz; }
            }
            __syncwarp();
        }
        // ---- a9: local energy at the end of the sweep (same terms as k_eloc_elec)
        double ksum = 0.0, psum = 0.0;
        for (int e = 0; e < ne; e++) {
            const int sp = e < s.ns[0] ? 0 : 1, p = sp ? e - s.ns[0] : e, ns = s.ns[sp];
            const double* A = As + sp * nsm * nsm;
            const double* Op = Os + ((sp * nsm + p) * 5) * nsm;
            double gx = 0, gy = 0, gz = 0, lp = 0;
            if (lane < ns) {
                const double aj = A[p * nsm + lane];
                gx = Op[nsm + lane] * aj; gy = Op[2 * nsm + lane] * aj; gz = Op[3 * nsm + lane] * aj; lp = Op[4 * nsm + lane] * aj;
            }
            const double rx = Rs[e], ry = Rs[nep + e], rz = Rs[2 * nep + e];
            double jx = 0, jy = 0, jz = 0, jl = 0, pot = 0;
            for (int k = lane; k < npart; k += 32) {
                Partner P = partner(s, Rs, nep, e, k);
                if (P.ok) {
                    const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
                    const double r = sqrt(dx * dx + dy * dy + dz * dz);
                    const double ir = 1.0 / r, iq = 1.0 / (1.0 + P.b * r);
                    const double du = P.a * iq * iq;
                    const double wgt = du * ir;
                    jx += wgt * dx; jy += wgt * dy; jz += wgt * dz;
                    jl += 2.0 * wgt - 2.0 * P.b * du * iq;
                    if (k >= ne) pot += P.a * ir;
                    else if (k > e) pot += ir;
                }
            }
            gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz); lp = warp_sum(lp);
            jx = warp_sum(jx); jy = warp_sum(jy); jz = warp_sum(jz); jl = warp_sum(jl); pot = warp_sum(pot);
            const double gg = gx * gx + gy * gy + gz * gz;
            const double tx = gx + jx, ty = gy + jy, tz = gz + jz;
            ksum += lp - gg + jl + (tx * tx + ty * ty + tz * tz);
            psum += pot;
        }
        const double K = -0.5 * ksum, e_new = K + (psum + s.e_nn);
        if (a.dmc) {  // row f1: tau_eff and the branching weight (same expressions as k_dmc_weight)
            const double te = dr2_all > 0.0 ? tau * dr2_acc / dr2_all : tau;
            const double arg = -te * ((e_old + e_new) / 2.0 - e_trial);
            weight *= exp(arg);
            if (lane == 0) wd.tau_eff[w] = te;
        }
        e_old = e_new;
        if (lane == 0) { wd.eloc[w] = e_new; wd.ekin[w] = K; }
    }
    // ---- shared memory -> HBM
    __syncwarp();
    for (int i = lane; i < 3 * nep; i += 32) wd.R[(long)w * 3 * nep + i] = Rs[i];
    for (int sp = 0; sp < 2; sp++) {
        const int ns = s.ns[sp], nsp = s.nsp[sp];
        for (int idx = lane; idx < ns * ns; idx += 32) {
            const int q = idx / ns, j = idx - q * ns;
            wd.AinvT[sp][((long)w * nsp + q) * nsp + j] = As[(sp * nsm + q) * nsm + j];
        }
        for (int idx = lane; idx < ns * 5 * ns; idx += 32) {
            const int q = idx / (5 * ns), rem = idx - q * 5 * ns, c = rem / ns, j = rem - c * ns;
            wd.Orb[sp][(((long)w * nsp + q) * 5 + c) * nsp + j] = Os[((sp * nsm + q) * 5 + c) * nsm + j];
        }
    }
    if (lane == 0) {
        wd.logpsi[w] = logpsi;
        if (a.dmc) { wd.weight[w] = weight; wd.eold[w] = e_old; }
        atomicAdd(&wd.stats[0], (unsigned long long)a.nsteps * ne);
        atomicAdd(&wd.stats[1], n_acc);
        atomicAdd(&wd.stats[2], n_tie);
        if (n_nonf) { atomicAdd(&wd.stats[3], n_nonf); wd.flags[w] = 1u; }
    }
}

}  // namespace qmc
