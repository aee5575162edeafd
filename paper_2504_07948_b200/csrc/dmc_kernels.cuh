// dmc_kernels.cuh -- row f1 of SURVEY 8(f): what turns the drift-diffusion sweep into a DMC generation.
// The paper runs fixed-node DMC (eq. 1; tau and population L131) and prints nothing about weights
// or branching; readings A28-A30 of DESIGN.md follow Umrigar, Nightingale, Runge, J. Chem. Phys. 99, 2865 (1993):
//   k_dmc_begin     E_old <- E_L, displacement sums <- 0 (start of a qmc_dmc_step call)
//   k_dmc_weight    tau_eff = tau * (accepted |sqrt(tau) chi|^2) / (proposed |sqrt(tau) chi|^2);
//                   weight *= exp(-tau_eff ((E_old + E_new)/2 - E_T));  E_old <- E_new
//   k_comb          fixed-population comb reconfiguration: W teeth (j + xi) W_tot / W over the cumulative weights,
//                   survivors stay in their slot, the k-th dead slot receives the k-th extra copy (donors ascending)
//   k_copy_walkers  the copies: positions, A^-1, row caches, scalars
// (the drift limiter itself and the displacement sums live in k_step).
#pragma once
#include "device_utils.cuh"

namespace qmc {

__global__ void k_dmc_begin(WalkDev wd) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= wd.W) return;
    wd.eold[w] = wd.eloc[w];
    wd.dr2[2 * w] = 0.0;
    wd.dr2[2 * w + 1] = 0.0;
}

// e_trial_dev != nullptr: the trial energy lives on the device (qmc_dmc_run: k_comb moves it between generations)
__global__ void k_dmc_weight(WalkDev wd, double tau, double e_trial, const double* e_trial_dev) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= wd.W) return;
    const double acc = wd.dr2[2 * w], all = wd.dr2[2 * w + 1];
    const double te = all > 0.0 ? tau * acc / all : tau;
    const double e_new = wd.eloc[w];
    if (e_trial_dev) e_trial = *e_trial_dev;
    const double arg = -te * ((wd.eold[w] + e_new) / 2.0 - e_trial);
    wd.weight[w] *= exp(arg);
    wd.eold[w] = e_new;
    wd.tau_eff[w] = te;
    wd.dr2[2 * w] = 0.0;
    wd.dr2[2 * w + 1] = 0.0;
}

struct CombOut {
    int* source;      // [W] slot j now holds a copy of old walker source[j]
    int* pair_dst;    // [W]
    int* pair_src;    // [W]
    int* n_pairs;     // [1]
    double* e_mixed;  // [1] sum w E_L / sum w before the reconfiguration
    int* mult;        // [W] scratch: multiplicities
    // population control of qmc_dmc_run (reading A32); all null / 0 for a plain qmc_branch
    double* e_trial_dev;  // [1] E_T <- e_mixed - feedback ln(W_tot / W)
    double feedback;
    double* branch_log;   // [3] of this reconfiguration: e_mixed, the new E_T, W_tot / W
};

// One CTA; the sums and the walk over the teeth are sequential in index order on purpose (one definite result).
__global__ void __launch_bounds__(256) k_comb(WalkDev wd, CombOut o, uint32_t step) {
    extern __shared__ double csm[];  // [W] weights (if they fit), else read from global
    const int W = wd.W, tid = threadIdx.x;
    const bool in_smem = (size_t)W * sizeof(double) <= 40 * 1024;
    const double* wts = wd.weight;
    if (in_smem) {
        for (int i = tid; i < W; i += blockDim.x) csm[i] = wd.weight[i];
        wts = csm;
    }
    for (int i = tid; i < W; i += blockDim.x) o.mult[i] = 0;
    __syncthreads();
    if (tid != 0) return;
    uint32_t out[4];
    philox4x32_10(0xFFFFFFFFu, step, 0xFFFFFFFFu, 3u, (uint32_t)(wd.seed & 0xFFFFFFFFull), (uint32_t)(wd.seed >> 32), out);
    const double xi = u01(out[0], out[1]);
    double tot = 0.0, ew = 0.0;
    for (int i = 0; i < W; i++) { tot = tot + wts[i]; ew += wts[i] * wd.eloc[i]; }
    o.e_mixed[0] = ew / tot;
    const double tooth = tot / (double)W;
    if (o.e_trial_dev) {
        const double et = ew / tot - o.feedback * log(tooth);
        o.e_trial_dev[0] = et;
        if (o.branch_log) { o.branch_log[0] = ew / tot; o.branch_log[1] = et; o.branch_log[2] = tooth; }
    }
    int i = 0;
    double cum = wts[0];
    for (int j = 0; j < W; j++) {
        const double t = ((double)j + xi) * tooth;
        while (i < W - 1 && !(t < cum)) { i++; cum = cum + wts[i]; }
        o.mult[i] += 1;
    }
    // survivors stay; the k-th dead slot takes the k-th extra copy, donors in ascending order
    int np = 0, donor = 0, left = 0;
    for (int k = 0; k < W; k++) {
        o.source[k] = k;
        if (o.mult[k] != 0) continue;
        if (left == 0) {
            while (o.mult[donor] < 2) donor++;
            left = o.mult[donor] - 1;
        }
        o.source[k] = donor;
        o.pair_dst[np] = k;
        o.pair_src[np] = donor;
        np++;
        left--;
        if (left == 0) donor++;
    }
    o.n_pairs[0] = np;
    for (int k = 0; k < W; k++) wd.weight[k] = tooth;
}

struct CopySeg { double* base; long per_walker; };  // per_walker doubles, a multiple of 2, 16-byte aligned
struct CopyArgs {
    CopySeg seg[5];
    int n_seg;
};

// grid (chunks, W): pair blockIdx.y copies its segments in 16-byte units, grid-stride over blockIdx.x
__global__ void __launch_bounds__(256) k_copy_walkers(WalkDev wd, CopyArgs a, CombOut o) {
    const int pr = blockIdx.y;
    if (pr >= o.n_pairs[0]) return;
    const int dst = o.pair_dst[pr], src = o.pair_src[pr];
    for (int sgi = 0; sgi < a.n_seg; sgi++) {
        const long n2 = a.seg[sgi].per_walker >> 1;
        const double2* s2 = reinterpret_cast<const double2*>(a.seg[sgi].base + (long)src * a.seg[sgi].per_walker);
        double2* d2 = reinterpret_cast<double2*>(a.seg[sgi].base + (long)dst * a.seg[sgi].per_walker);
        for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (long)gridDim.x * blockDim.x) d2[i] = s2[i];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        wd.logpsi[dst] = wd.logpsi[src];
        wd.sign[dst] = wd.sign[src];
        wd.flags[dst] = wd.flags[src];
        wd.eloc[dst] = wd.eloc[src];
        wd.ekin[dst] = wd.ekin[src];
        wd.eold[dst] = wd.eold[src];
        wd.tau_eff[dst] = wd.tau_eff[src];
    }
}

}  // namespace qmc
