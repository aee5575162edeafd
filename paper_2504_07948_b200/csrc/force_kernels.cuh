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

}  // namespace qmc
