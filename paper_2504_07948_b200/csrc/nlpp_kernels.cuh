// nlpp_kernels.cuh -- row f3 of SURVEY 8(f): the non-local pseudopotential energy by spherical quadrature (PAPER.md L129
// "ccECP pseudopotentials", L180 "the non-local pseudopotential contribution"; reading A34).  Atom I carries
// channels l (0..2) with v_l(r) = beta exp(-alpha r^2), cut at rcut_I; for every electron i with r = |r_i - R_I| < rcut_I
//   (V_nl Psi / Psi)_iI = sum_q w_q [ sum_l (2l+1) v_l(r) P_l(cos th_q) ] Psi(.., r_q, ..) / Psi(.., r_i, ..),
//   r_q = R_I + r O_q,  O_q = Rot * icosahedron vertex q,  w_q = 1/12,  cos th_q = O_q . (r_i - R_I) / r,
// Rot a uniform random rotation per (walker, step, electron) from Philox blocks 4 and 5.  These are "ratio-only" moves:
// stages a3-a6 of the sweep (basis values, MO contraction, determinant ratio against the row of A^-T, Jastrow ratio)
// without accept or update, twelve points per (electron, atom) pair -- so the points of all walkers are batched through
// the same k_basis (values only) and k_mo_streamk as the sweep.
//   k_nl_count / k_nl_scan / k_nl_fill   the (walker, electron, atom) pairs inside the cut-offs, in a definite order
//   k_nl_points                          the 12 points of every pair and their angular factors
//   k_nl_ratio                           one CTA per point: determinant ratio x exp(Jastrow difference) x angular factor
//   k_nl_reduce                          fixed-order sum per walker
#pragma once
#include "device_utils.cuh"

namespace qmc {

__device__ __forceinline__ bool nl_in_range(const SysDev& s, int I, double dx, double dy, double dz, double* r_out) {
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    *r_out = r;
    return s.ecp_off[I + 1] > s.ecp_off[I] && r < s.ecp_rcut[I];
}

// one thread per (walker, electron of the spin)
__global__ void __launch_bounds__(256) k_nl_count(SysDev s, WalkDev wd, NlArgs a) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)wd.W * a.ns) return;
    const int w = (int)(idx / a.ns), e = a.e0 + (int)(idx % a.ns);
    const double* Rw = wd.R + (long)w * 3 * wd.nep;
    const double rx = Rw[e], ry = Rw[wd.nep + e], rz = Rw[2 * wd.nep + e];
    int c = 0;
    for (int I = 0; I < s.n_atoms; I++) {
        double r;
        if (nl_in_range(s, I, rx - s.atom_xyz[3 * I], ry - s.atom_xyz[3 * I + 1], rz - s.atom_xyz[3 * I + 2], &r)) c++;
    }
    a.cnt[idx] = c;
}

// exclusive scan of cnt[0..n) in place, cnt[n] = total.  One CTA of 1024 threads, each owning a contiguous chunk.
__global__ void __launch_bounds__(1024) k_nl_scan(int* cnt, long n) {
    __shared__ int part[1024];
    const int tid = threadIdx.x;
    const long chunk = (n + 1023) / 1024, lo = tid * chunk, hi = lo + chunk < n ? lo + chunk : n;
    int sum = 0;
    for (long i = lo; i < hi; i++) sum += cnt[i];
    part[tid] = sum;
    __syncthreads();
    if (tid == 0) {
        int acc = 0;
        for (int i = 0; i < 1024; i++) { const int v = part[i]; part[i] = acc; acc += v; }
        cnt[n] = acc;
    }
    __syncthreads();
    int acc = part[tid];
    for (long i = lo; i < hi; i++) { const int v = cnt[i]; cnt[i] = acc; acc += v; }
}

__global__ void __launch_bounds__(256) k_nl_fill(SysDev s, WalkDev wd, NlArgs a) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)wd.W * a.ns) return;
    const int w = (int)(idx / a.ns), e = a.e0 + (int)(idx % a.ns);
    const double* Rw = wd.R + (long)w * 3 * wd.nep;
    const double rx = Rw[e], ry = Rw[wd.nep + e], rz = Rw[2 * wd.nep + e];
    int o = a.cnt[idx];
    for (int I = 0; I < s.n_atoms; I++) {
        double r;
        if (nl_in_range(s, I, rx - s.atom_xyz[3 * I], ry - s.atom_xyz[3 * I + 1], rz - s.atom_xyz[3 * I + 2], &r)) {
            a.pair_w[o] = w; a.pair_e[o] = e; a.pair_I[o] = I;
            o++;
        }
    }
}

// vertex q = 4 c + 2 a + b: coordinate c is 0, coordinate c+1 is (+/-) n, coordinate c+2 is (+/-) phi n
__device__ __forceinline__ void icosahedron_vertex(int q, double v[3]) {
    const double phi = (1.0 + sqrt(5.0)) / 2.0;
    const double n = 1.0 / sqrt(1.0 + phi * phi);
    const int c = q / 4, sa = (q / 2) % 2, sb = q % 2;
    v[c] = 0.0;
    v[(c + 1) % 3] = sa ? -n : n;
    v[(c + 2) % 3] = sb ? -phi * n : phi * n;
}

// one thread per (pair, q)
__global__ void __launch_bounds__(256) k_nl_points(SysDev s, WalkDev wd, NlArgs a, int n_pairs) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)n_pairs * 12) return;
    const int pr = (int)(idx / 12), q = (int)(idx % 12);
    const int w = a.pair_w[pr], e = a.pair_e[pr], I = a.pair_I[pr];
    const double* Rw = wd.R + (long)w * 3 * wd.nep;
    const double ax = s.atom_xyz[3 * I], ay = s.atom_xyz[3 * I + 1], az = s.atom_xyz[3 * I + 2];
    const double dx = Rw[e] - ax, dy = Rw[wd.nep + e] - ay, dz = Rw[2 * wd.nep + e] - az;
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    // uniform random rotation (Shoemake): three uniforms -> unit quaternion -> matrix
    const uint32_t k0 = (uint32_t)(wd.seed & 0xFFFFFFFFull), k1 = (uint32_t)(wd.seed >> 32);
    uint32_t o4[4], o5[4];
    philox4x32_10(wd.first_walker + (uint32_t)w, a.step, (uint32_t)e, 4u, k0, k1, o4);
    philox4x32_10(wd.first_walker + (uint32_t)w, a.step, (uint32_t)e, 5u, k0, k1, o5);
    const double u1 = u01(o4[0], o4[1]), u2 = u01(o4[2], o4[3]), u3 = u01(o5[0], o5[1]);
    const double TWO_PI = 6.283185307179586476925286766559;
    const double qa = sqrt(1.0 - u1), qb = sqrt(u1);
    const double x = qa * sin(TWO_PI * u2), y = qa * cos(TWO_PI * u2), z = qb * sin(TWO_PI * u3), ww = qb * cos(TWO_PI * u3);
    double rot[9];
    rot[0] = 1.0 - 2.0 * (y * y + z * z); rot[1] = 2.0 * (x * y - z * ww);       rot[2] = 2.0 * (x * z + y * ww);
    rot[3] = 2.0 * (x * y + z * ww);       rot[4] = 1.0 - 2.0 * (x * x + z * z); rot[5] = 2.0 * (y * z - x * ww);
    rot[6] = 2.0 * (x * z - y * ww);       rot[7] = 2.0 * (y * z + x * ww);       rot[8] = 1.0 - 2.0 * (x * x + y * y);
    double v[3], od[3];
    icosahedron_vertex(q, v);
#pragma unroll
    for (int d = 0; d < 3; d++) od[d] = rot[3 * d] * v[0] + rot[3 * d + 1] * v[1] + rot[3 * d + 2] * v[2];
    a.pts[3 * idx] = ax + r * od[0];
    a.pts[3 * idx + 1] = ay + r * od[1];
    a.pts[3 * idx + 2] = az + r * od[2];
    const double c = (od[0] * dx + od[1] * dy + od[2] * dz) / r;
    double vl[3] = {0.0, 0.0, 0.0};  // (2l+1) v_l(r)
    for (int ch = s.ecp_off[I]; ch < s.ecp_off[I + 1]; ch++) {
        const int l = s.ecp_l[ch];
        vl[l] += (double)(2 * l + 1) * s.ecp_beta[ch] * exp(-s.ecp_alpha[ch] * r * r);
    }
    a.ang[idx] = (vl[0] + vl[1] * c + vl[2] * (1.5 * c * c - 0.5)) / 12.0;
}

// one 128-thread CTA per point of the chunk [pt0, pt0 + n): V [n][ldv] holds the orbital values at the points
// (a warp per point leaves the GPU with 8 warps per SM on a 5 W chunk: latency-bound, 71 us against 20)
constexpr int NL_RATIO_THREADS = 128;
__global__ void __launch_bounds__(NL_RATIO_THREADS) k_nl_ratio(SysDev s, WalkDev wd, NlArgs a, long pt0, int n, const double* __restrict__ V) {
    __shared__ double red[2 * (NL_RATIO_THREADS / 32)];
    const int t = blockIdx.x, tid = threadIdx.x;
    const long gp = pt0 + t;
    const int pr = (int)(gp / 12);
    const int w = a.pair_w[pr], e = a.pair_e[pr], p = e - a.e0;
    const int nsp = s.nsp[a.spin], nep = wd.nep;
    const double* arow = wd.AinvT[a.spin] + ((long)w * nsp + p) * nsp;
    const double* vrow = V + (long)t * wd.ldv;
    double acc[2] = {0.0, 0.0};  // determinant ratio, Jastrow difference
    for (int j = tid; j < a.ns; j += NL_RATIO_THREADS) acc[0] += vrow[j] * arow[j];
    const double* Rw = wd.R + (long)w * 3 * nep;
    const double rx = Rw[e], ry = Rw[nep + e], rz = Rw[2 * nep + e];
    const double qx = a.pts[3 * gp], qy = a.pts[3 * gp + 1], qz = a.pts[3 * gp + 2];
    const int npart = s.ne + s.n_atoms;
    for (int k = tid; k < npart; k += NL_RATIO_THREADS) {
        Partner P = partner(s, Rw, nep, e, k);
        if (P.ok) {
            const double dx = rx - P.x, dy = ry - P.y, dz = rz - P.z;
            const double ex = qx - P.x, ey = qy - P.y, ez = qz - P.z;
            const double r0 = sqrt(dx * dx + dy * dy + dz * dz), r1 = sqrt(ex * ex + ey * ey + ez * ez);
            // u(r1) - u(r0) = a (r1 - r0) / ((1 + b r1)(1 + b r0))
            acc[1] += P.a * (r1 - r0) / ((1.0 + P.b * r1) * (1.0 + P.b * r0));
        }
    }
    block_sum<NL_RATIO_THREADS, 2>(acc, red);
    if (tid == 0) a.terms[gp] = a.ang[gp] * acc[0] * exp(acc[1]);
}

// one CTA per walker: its pairs are contiguous (offsets cnt[w * ns] .. cnt[(w + 1) * ns]); fixed-shape sum
__global__ void __launch_bounds__(256) k_nl_reduce(WalkDev wd, NlArgs a, double* __restrict__ vnl) {
    __shared__ double red[8];
    const int w = blockIdx.x;
    const long lo = 12L * a.cnt[(long)w * a.ns], hi = 12L * a.cnt[(long)(w + 1) * a.ns];
    double acc[1] = {0.0};
    for (long i = lo + threadIdx.x; i < hi; i += 256) acc[0] += a.terms[i];
    block_sum<256, 1>(acc, red);
    if (threadIdx.x == 0) vnl[w] += acc[0];
}

}  // namespace qmc
