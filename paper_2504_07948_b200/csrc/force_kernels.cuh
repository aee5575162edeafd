// force_kernels.cuh -- row f2 of SURVEY 8(f), first half: d ln|Psi| / d R_a for every atom and walker, the wave-function
// ("Pulay") term of a QMC force estimator.  The paper's eq. (3), d ln D / d lambda = tr(A^-1 dA/d lambda),
// with lambda a nuclear coordinate: basis functions move with their nucleus, dPhi_l/dR_a = -grad Phi_l for l on a, so
//   d ln D / d R_a = - sum_p sum_{l on a} grad Phi_l(r_p) (C A^-1)[l][p]          (both spins added)
// plus the electron-nucleus Jastrow term  - sum_i u_en'(r_ia) (r_i - R_a) / r_ia.
// (C A^-1)^T = A^-T C^T is one batched FP64 DMMA GEMM per spin (2 N_s^2 N_b flop per walker -- the O(N^3) part the paper
// batches over walkers, L184); k_dlogpsi then needs only the shells of one atom per CTA.  The derivative of E_L itself
// (eq. 4) is not built.
#pragma once
#include "device_utils.cuh"

namespace qmc {

__global__ void k_plain_C(const double* __restrict__ in, int nb, int ns, double* __restrict__ Cp, int nsp, const int* __restrict__ fmap) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)nb * ns) return;
    const int l = (int)(idx / ns), j = (int)(idx % ns);
    Cp[(long)fmap[l] * nsp + j] = in[idx];
}

// grid (n_atoms, W), 128 threads: threads stride over the electrons of the spin; fixed-shape reduction at the end
__global__ void __launch_bounds__(128) k_dlogpsi(SysDev s, WalkDev wd, int spin, const double* __restrict__ Mt /* [W][nsp][nbp] */,
                                                 double* __restrict__ acc /* [W][n_atoms][3] */, int with_jastrow) {
    __shared__ double red[3 * 4];
    const int a = blockIdx.x, w = blockIdx.y, tid = threadIdx.x;
    const int ns = s.ns[spin], nsp = s.nsp[spin], nep = wd.nep, e0 = spin == 0 ? 0 : s.ns[0];
    const double* Rw = wd.R + (long)w * 3 * nep;
    const int sh0 = s.atom_shell_off[a], sh1 = s.atom_shell_off[a + 1];
    double f3[3] = {0.0, 0.0, 0.0};
    for (int p = tid; p < ns; p += 128) {
        const double rx = Rw[e0 + p], ry = Rw[nep + e0 + p], rz = Rw[2 * nep + e0 + p];
        const double* m = Mt + ((long)w * nsp + p) * s.nbp;
        for (int q = sh0; q < sh1; q++) {
            const ShellRec rec = s.shells[s.atom_shell_list[q]];
            const double x = rx - rec.x, y = ry - rec.y, z = rz - rec.z;
            const double t = x * x + y * y + z * z;
            double g = 0.0, g1 = 0.0;
            for (int k = 0; k < rec.nprim; k++) {
                const double al = __ldg(s.alpha + rec.poff + k);
                const double e = __ldg(s.coef + rec.poff + k) * exp(-al * t);
                g += e;
                g1 -= al * e;
            }
            const double tg1 = 2.0 * g1;
            auto add = [&](int mm, double S, double Sx, double Sy, double Sz) {  // grad Phi = g grad S + 2 g' S x
                const double c = m[rec.f0 + mm];
                f3[0] -= (g * Sx + tg1 * S * x) * c;
                f3[1] -= (g * Sy + tg1 * S * y) * c;
                f3[2] -= (g * Sz + tg1 * S * z) * c;
            };
            const double s3 = 1.7320508075688772;
            if (rec.l == 0) {
                add(0, 1.0, 0.0, 0.0, 0.0);
            } else if (rec.l == 1) {
                add(0, x, 1.0, 0.0, 0.0);
                add(1, y, 0.0, 1.0, 0.0);
                add(2, z, 0.0, 0.0, 1.0);
            } else {
                add(0, s3 * x * y, s3 * y, s3 * x, 0.0);
                add(1, s3 * y * z, 0.0, s3 * z, s3 * y);
                add(2, z * z - 0.5 * (x * x + y * y), -x, -y, 2.0 * z);
                add(3, s3 * x * z, s3 * z, 0.0, s3 * x);
                add(4, (0.5 * s3) * (x * x - y * y), s3 * x, -s3 * y, 0.0);
            }
        }
    }
    if (with_jastrow) {  // - sum_i u_en'(r_ia) (r_i - R_a) / r_ia, u_en = -Z r / (1 + b r)
        const double ax = s.atom_xyz[3 * a], ay = s.atom_xyz[3 * a + 1], az = s.atom_xyz[3 * a + 2], Za = s.atom_Z[a];
        for (int i = tid; i < s.ne; i += 128) {
            const double dx = Rw[i] - ax, dy = Rw[nep + i] - ay, dz = Rw[2 * nep + i] - az;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double du = pade_du(-Za, s.b_en, r);
            f3[0] -= du * dx / r; f3[1] -= du * dy / r; f3[2] -= du * dz / r;
        }
    }
    block_sum<128, 3>(f3, red);
    if (tid == 0) {
        double* o = acc + ((long)w * s.n_atoms + a) * 3;
        o[0] += f3[0]; o[1] += f3[1]; o[2] += f3[2];
    }
}

// ------------------------------------------------------------------------------------------------
// Row f2, second half: d E_L / d R_a by the paper's eq. (4),
//   dE_L/dR_a = sum_spin tr(A^-1 dB/dR_a - X dA/dR_a) + sum_i dc_i/dR_a + dV/dR_a,   X = A^-1 B A^-1,
//   B[i][j] = -1/2 [ lap phi_j(r_i) + 2 gJ_i . grad phi_j(r_i) ],  c_i = -1/2 [ lap_i J + |gJ_i|^2 ]      (A33).
// With Mt[i][l] = (C A^-1)[l][i] and Nt[i][l] = (C X)[l][i] (batched DMMA GEMMs over walkers, the O(N^3) part) the traces
// collapse to sums over the functions of atom a alone:
//   tr(A^-1 dB - X dA)_d = sum_i sum_{l on a} [ T_d,l(r_i) Mt[i][l] + d_d Phi_l(r_i) Nt[i][l] ]  -  sum_i dgJ_i . G_i,
//   T_d,l = 1/2 d_d lap Phi_l + sum_b gJ_i,b d_d d_b Phi_l,    G_i = sum_j grad phi_j(r_i) A^-1[j][i],
//   dgJ_i,b = -d_d d_b u_en(|r_i - R_a|).
// k_force_prep: one warp per electron -- gJ_i, G_i and row i of B.   k_deloc: one CTA per (atom, walker).

// fg [W][ne][8] = gJ (3), G (3), 2 unused;  Bm [W][nsp][nsp] per spin (rows / columns >= ns stay zero)
__global__ void __launch_bounds__(256, 4) k_force_prep(SysDev s, WalkDev wd, double* __restrict__ fg, double* __restrict__ Bm0,
                                                       double* __restrict__ Bm1) {
    const int w = blockIdx.y;
    const int e = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (e >= s.ne) return;
    const int spin = e < s.ns[0] ? 0 : 1, p = spin ? e - s.ns[0] : e;
    const int ns = s.ns[spin], nsp = s.nsp[spin], nep = wd.nep;
    const double* arow = wd.AinvT[spin] + ((long)w * nsp + p) * nsp;
    const double* orb = wd.Orb[spin] + ((long)w * nsp + p) * 5 * nsp;
    // the Jastrow gradient first (it does not need the row caches), then ONE pass over the cached rows for G_i and row i of B
    const double* Rw = wd.R + (long)w * 3 * nep;
    const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
    double jx = 0, jy = 0, jz = 0;
    const int npart = s.ne + s.n_atoms;
    for (int k = lane; k < npart; k += 32) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double wgt = pade_du(P.a, P.b, r) / r;
            jx += wgt * dx; jy += wgt * dy; jz += wgt * dz;
        }
    }
    jx = warp_sum(jx); jy = warp_sum(jy); jz = warp_sum(jz);
    double* brow = (spin ? Bm1 : Bm0) + ((long)w * nsp + p) * nsp;
    double gx = 0, gy = 0, gz = 0;
    for (int j = lane; j < ns; j += 32) {
        const double a = arow[j];
        const double o1 = orb[nsp + j], o2 = orb[2 * nsp + j], o3 = orb[3 * nsp + j];
        gx += o1 * a; gy += o2 * a; gz += o3 * a;
        brow[j] = -0.5 * (orb[4 * nsp + j] + 2.0 * (jx * o1 + jy * o2 + jz * o3));
    }
    gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz);
    if (lane == 0) {
        double* o = fg + ((long)w * s.ne + e) * 8;
        o[0] = jx; o[1] = jy; o[2] = jz; o[3] = gx; o[4] = gy; o[5] = gz;
    }
}

// grid (n_atoms, W), 128 threads.  spin 0 / 1: the trace terms of that spin (threads stride over its electrons);
// with_rest: also - sum_i dgJ_i . G_i + sum_i dc_i + dV (all electrons, both spins).
// acc_psi != nullptr: d ln|Psi| / d R_a (what k_dlogpsi computes) from the same radial sums, in the same order.
__global__ void __launch_bounds__(128) k_deloc(SysDev s, WalkDev wd, int spin, const double* __restrict__ Mt, const double* __restrict__ Nt,
                                               const double* __restrict__ fg, double* __restrict__ acc, double* __restrict__ acc_psi,
                                               int with_rest) {
    __shared__ double red[6 * 4];
    const int a = blockIdx.x, w = blockIdx.y, tid = threadIdx.x;
    const int ns = s.ns[spin], nsp = s.nsp[spin], nep = wd.nep, e0 = spin == 0 ? 0 : s.ns[0];
    const double* Rw = wd.R + (long)w * 3 * nep;
    const int sh0 = s.atom_shell_off[a], sh1 = s.atom_shell_off[a + 1];
    double f3[3] = {0.0, 0.0, 0.0}, p3[3] = {0.0, 0.0, 0.0};
    for (int p = tid; p < ns; p += 128) {
        const double rx = Rw[e0 + p], ry = Rw[nep + e0 + p], rz = Rw[2 * nep + e0 + p];
        const double* m = Mt + ((long)w * nsp + p) * s.nbp;
        const double* n = Nt + ((long)w * nsp + p) * s.nbp;
        const double* gj = fg + ((long)w * s.ne + e0 + p) * 8;
        const double jx = gj[0], jy = gj[1], jz = gj[2];
        for (int q = sh0; q < sh1; q++) {
            const ShellRec rec = s.shells[s.atom_shell_list[q]];
            const double x = rx - rec.x, y = ry - rec.y, z = rz - rec.z;
            const double t = x * x + y * y + z * z;
            double g = 0.0, g1 = 0.0, g2 = 0.0, g3 = 0.0;
            for (int k = 0; k < rec.nprim; k++) {
                const double al = __ldg(s.alpha + rec.poff + k);
                const double e = __ldg(s.coef + rec.poff + k) * exp(-al * t);
                g += e;
                g1 -= al * e;
                g2 += al * al * e;
                g3 -= al * al * al * e;
            }
            const double h = (double)(4 * rec.l + 6) * g1 + 4.0 * t * g2;     // lap Phi = S h
            const double h1 = (double)(4 * rec.l + 10) * g2 + 4.0 * t * g3;   // dh/dt
            const double xg = x * jx + y * jy + z * jz;
            // S, grad S, (Hessian of S) . gJ
            auto add = [&](int mm, double S, double Sx, double Sy, double Sz, double Hx, double Hy, double Hz) {
                const double cm = m[rec.f0 + mm], cn = n[rec.f0 + mm];
                const double dsg = Sx * jx + Sy * jy + Sz * jz;
                const double k1 = 0.5 * h + 2.0 * g1 * xg;                 // multiplies grad S
                const double k2 = S * (h1 + 4.0 * g2 * xg) + 2.0 * g1 * dsg;  // multiplies x
                const double k3 = 2.0 * g1 * S;                            // multiplies gJ
                const double tg1 = 2.0 * g1 * S;
                f3[0] += (k1 * Sx + k2 * x + k3 * jx + g * Hx) * cm + (g * Sx + tg1 * x) * cn;
                f3[1] += (k1 * Sy + k2 * y + k3 * jy + g * Hy) * cm + (g * Sy + tg1 * y) * cn;
                f3[2] += (k1 * Sz + k2 * z + k3 * jz + g * Hz) * cm + (g * Sz + tg1 * z) * cn;
                p3[0] -= (g * Sx + tg1 * x) * cm;
                p3[1] -= (g * Sy + tg1 * y) * cm;
                p3[2] -= (g * Sz + tg1 * z) * cm;
            };
            const double s3 = 1.7320508075688772;
            if (rec.l == 0) {
                add(0, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0);
            } else if (rec.l == 1) {
                add(0, x, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0);
                add(1, y, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0);
                add(2, z, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0);
            } else {
                add(0, s3 * x * y, s3 * y, s3 * x, 0.0, s3 * jy, s3 * jx, 0.0);
                add(1, s3 * y * z, 0.0, s3 * z, s3 * y, 0.0, s3 * jz, s3 * jy);
                add(2, z * z - 0.5 * (x * x + y * y), -x, -y, 2.0 * z, -jx, -jy, 2.0 * jz);
                add(3, s3 * x * z, s3 * z, 0.0, s3 * x, s3 * jz, 0.0, s3 * jx);
                add(4, (0.5 * s3) * (x * x - y * y), s3 * x, -s3 * y, 0.0, s3 * jx, -s3 * jy, 0.0);
            }
        }
    }
    if (with_rest) {
        const double ax = s.atom_xyz[3 * a], ay = s.atom_xyz[3 * a + 1], az = s.atom_xyz[3 * a + 2], Za = s.atom_Z[a];
        const double A = -Za, b = s.b_en;
        for (int i = tid; i < s.ne; i += 128) {
            const double* gj = fg + ((long)w * s.ne + i) * 8;
            const double vx = gj[0] + gj[3], vy = gj[1] + gj[4], vz = gj[2] + gj[5];   // gJ_i + G_i
            const double dx = Rw[i] - ax, dy = Rw[nep + i] - ay, dz = Rw[2 * nep + i] - az;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double ir = 1.0 / r, iq = 1.0 / (1.0 + b * r);
            const double u1 = A * iq * iq, u2 = -2.0 * b * u1 * iq, u3 = -3.0 * b * u2 * iq;
            // -dgJ . v = (u2/r^2 - u1/r^3) x_d (x . v) + u1 v_d / r ;  dc_i = 1/2 (u3 + 2 u2/r - 2 u1/r^2) x_d / r + (-dgJ . gJ)
            const double xv = dx * vx + dy * vy + dz * vz;
            const double c1 = (u2 - u1 * ir) * ir * ir * xv + (0.5 * (u3 + 2.0 * u2 * ir - 2.0 * u1 * ir * ir) - Za * ir * ir) * ir;
            const double c2 = u1 * ir;
            f3[0] += c1 * dx + c2 * vx; f3[1] += c1 * dy + c2 * vy; f3[2] += c1 * dz + c2 * vz;
            p3[0] -= c2 * dx; p3[1] -= c2 * dy; p3[2] -= c2 * dz;   // - u_en'(r) (r_i - R_a) / r
        }
        for (int bb = tid; bb < s.n_atoms; bb += 128) {
            if (bb == a) continue;
            const double yx = ax - s.atom_xyz[3 * bb], yy = ay - s.atom_xyz[3 * bb + 1], yz = az - s.atom_xyz[3 * bb + 2];
            const double r2 = yx * yx + yy * yy + yz * yz;
            const double c = -Za * s.atom_Z[bb] / (r2 * sqrt(r2));
            f3[0] += c * yx; f3[1] += c * yy; f3[2] += c * yz;
        }
    }
    double f6[6] = {f3[0], f3[1], f3[2], p3[0], p3[1], p3[2]};
    block_sum<128, 6>(f6, red);
    if (tid == 0) {
        double* o = acc + ((long)w * s.n_atoms + a) * 3;
        o[0] += f6[0]; o[1] += f6[1]; o[2] += f6[2];
        if (acc_psi) {
            double* q = acc_psi + ((long)w * s.n_atoms + a) * 3;
            q[0] += f6[3]; q[1] += f6[4]; q[2] += f6[5];
        }
    }
}

}  // namespace qmc
