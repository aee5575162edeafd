// qmc_internal.cuh -- device-side data layout shared by the kernels and the host scheduler.
//
// HBM layout (all FP64 unless noted; "NSP" = n_s rounded up to 16, "NBP" = n_basis rounded up to 32 = 32 KB,
// padding is zero and stays zero, so padded orbitals/functions contribute nothing):
//   CT[s]     [NT][KB][32][132]     MO coefficients of spin s, pre-tiled as the B stages of the stream-K GEMM
//                                   (tile = 32 basis functions x 128 orbitals, rows padded to 132 doubles)
//   R         [W][3][NEP]           positions, walker-major SoA (coalesced over electrons inside a walker)
//   AinvT[s]  [W][NSP][NSP]         AinvT[p][j] = (A^-1)[j][p]: row p is the column the ratio needs (A18)
//   Orb[s]    [W][NSP(p)][5][NSP]   value / d/dx / d/dy / d/dz / laplacian of the orbitals at the CURRENT
//                                   position of electron p (row cache: drift and E_L cost O(N_s) per electron)
//   PhiT      [MT][KB][128][36]     basis functions at the proposed positions, pre-tiled as the A stages
//                                   (row = walker*5 + component, tile = 128 rows x 32 functions, padded to 36)
//   V         [W*5][LDV]            orbital rows at the proposed positions (GEMM output)
//   window    Vbuf,Wbuf,W2 [W][KP][NSP], SinvT [W][KP][KP], YT [W][NSP][KP], plist [W][KP] int, mcount [W] int
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmc {

struct ShellRec {
    double x, y, z;
    int l, f0, nprim, poff;
};

// One shell as the basis kernel reads it: a self-contained 96-byte record (six 16-byte loads, no dependent
// second load for the primitives).  Up to three primitives are inline (unused slots have coef 0, alpha 0 and
// contribute exactly 0); primitives beyond three are read from alpha/coef at poff + 3.
struct __align__(16) KbShell {
    double x, y, z;
    double a[3];
    double c[3];
    int l, f0, nprim, poff;
    double pad;
};

struct SysDev {
    int n_atoms, n_shells, n_basis, nbp, kb;  // kb = nbp / 32
    int ns[2], nsp[2], ne;
    const double* atom_xyz;  // [n_atoms][3]
    const double* atom_Z;
    const ShellRec* shells;
    const int4* kb_counts;  // [kb]: number of s, p, d shells owning a function of k-block kb (32 functions), list offset
    const KbShell* kb_list; // shells of every k-block, grouped s | p | d (a shell may be in two blocks)
    const int* win_items;   // window kernel: the occupied slots (kb * 32 + slot) of kb_list, those of the k-blocks below kb/2
    int n_win_items, n_win_first;  //   first (n_win_first of them), each half ordered s | p | d
    const int* fmap;        // [n_basis] caller's function index -> internal one (shells grouped by reach, Morton-ordered)
    const double* Cplain[2];   // [nbp][nsp] MO coefficients, internal function order, plain row-major (row f2: C A^-1)
    const int* atom_shell_off; // [n_atoms + 1] shells of every atom in atom_shell_list
    const int* atom_shell_list;
    const double* alpha;
    const double* coef;
    const double* CT[2];  // tiled, see mo_streamk.cuh
    int nt[2];            // 128-column tiles per spin
    double a_anti, a_para, b_ee, b_en;
    double e_nn;  // nuclear repulsion
    // row f3 (qmc_set_ecp; all null until then): channels grouped by atom, ecp_off [n_atoms + 1]
    const int* ecp_off;
    const int* ecp_l;
    const double* ecp_beta;
    const double* ecp_alpha;
    const double* ecp_rcut;  // [n_atoms]
};

struct WalkDev {
    int W, ne, nep, ldv, kp;
    int onepass;   // QMC_STEP_ONEPASS: the one-pass step kernel whatever the row length
    int lean;   // this set of walkers is one LANE of a crowd (its kernels share the SMs with the other lane's contraction)
    double* R;
    double* AinvT[2];
    double* Orb[2];
    double* Phi;  // tiled PhiT
    int mt;       // 128-row tiles of Phi
    double* V;
    double* mo_ws;       // stream-K partial tiles [n_sm][128*128]
    unsigned* mo_flags;  // [n_sm]
    int mo_grid;
    double *Vbuf, *Wbuf, *W2, *SinvT, *YT, *bvec, *cvec, *xcol;
    int *plist, *mcount;
    double *rp, *G, *u, *dJ, *gJn;  // per-walker proposal scalars: [W][3], [W][3], [W], [W], [W][3]
    double* logpsi;
    int* sign;
    unsigned* flags;  // sticky non-finite flag per walker
    double *eloc, *ekin, *ebuf;  // ebuf [W][ne][2]
    uint8_t* bits;               // [T][ne][W] of the current sweep call
    double *ratio_log, *pacc_log;
    unsigned long long* stats;  // proposed, accepted, ties, nonfinite
    uint64_t seed;
    uint32_t first_walker;
    // DMC generation (row f1): drift-limiter constant (<= 0: off), per-walker weight, E_L at the start of the generation,
    // sums of |sqrt(tau) chi|^2 over accepted / all proposals [W][2], the pending proposal's value [W], tau_eff [W]
    double lim_a;
    double *weight, *eold, *dr2, *dr2p, *tau_eff;
    // optional screening of the MO contraction (QMC_SCREEN_MO): A stages whose largest |entry| is below screen_theta are
    // not contracted.  tilemax [MT][KB] from k_basis; plan_* from k_mo_plan (see mo_streamk.cuh); mo_work [2]: executed
    // and dense (tile, k-block) iterations since creation.  screen_theta < 0: off, the plan is not used.
    double screen_theta;
    double* tilemax;
    int *plan_cnt, *plan_pre, *plan_kb;
    unsigned long long* mo_work;
};

// row f3 (nlpp_kernels.cuh): one spin of one qmc_get_vnl call
struct NlArgs {
    int spin, e0, ns;        // electrons e0 .. e0 + ns - 1
    int* cnt;                // [W * ns + 1] pairs of (w, p); after the scan: offsets, cnt[W * ns] = total
    int* pair_w;             // [n_pairs]
    int* pair_e;             // global electron index
    int* pair_I;
    double* pts;             // [n_pairs * 12][3]
    double* ang;             // [n_pairs * 12] sum_l (2l+1) v_l(r) P_l(cos th_q) / 12
    double* terms;           // [n_pairs * 12] ang * ratio
    uint32_t step;
};

}  // namespace qmc
