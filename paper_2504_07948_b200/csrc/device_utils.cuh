// device_utils.cuh -- small device helpers shared by the kernels: fixed-shape reductions, Philox4x32-10 and the
// uniform mapping (reading A11), the Pade Jastrow terms (reading A5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qmc_internal.cuh"

namespace qmc {

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
// Pade Jastrow pieces
__device__ __forceinline__ double pade_u(double a, double b, double r) { return a * r / (1.0 + b * r); }
__device__ __forceinline__ double pade_du(double a, double b, double r) { double q = 1.0 + b * r; return a / (q * q); }
__device__ __forceinline__ double pade_d2u(double a, double b, double r) { double q = 1.0 + b * r; return -2.0 * a * b / (q * q * q); }

// partner k of electron e: k < ne electrons (skip k == e), then atoms
struct Partner { double x, y, z, a, b; bool ok; };
__device__ __forceinline__ Partner partner(const SysDev& s, const double* Rw, int nep, int e, int k) {
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

}  // namespace qmc
