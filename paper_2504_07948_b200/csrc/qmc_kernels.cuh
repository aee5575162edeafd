// qmc_kernels.cuh -- launchers of the kernels in qmc_kernels.cu (host-side scheduler interface).
#pragma once
#include "qmc_internal.cuh"

namespace qmc {

// tilemax ([MT][KB], may be NULL): max |entry| of every A stage, for the optional screening of the MO contraction
cudaError_t launch_basis(const SysDev& s, const double* pts, int n_points, double* PhiT, double* tilemax, cudaStream_t st);
cudaError_t launch_basis_values(const SysDev& s, const double* pts, int n_points, double* PhiT, cudaStream_t st);
cudaError_t launch_mo(const SysDev& s, int spin, const double* PhiT, int rows, double* V, long ldv, double* ws, unsigned* flags,
                      int grid, unsigned epoch, const WalkDev* plan, cudaStream_t st, unsigned long long* trace = nullptr);
cudaError_t launch_mo_plan(const SysDev& s, int spin, const WalkDev& wd, int rows, cudaStream_t st);
int mo_grid_for(const SysDev& s, int spin, int rows, int n_sm);
size_t mo_ws_bytes(int grid);
size_t phiT_bytes(const SysDev& s, int rows);
cudaError_t launch_tile_C(const double* in, int nb, int ns, double* CT, int kb, const int* fmap, cudaStream_t st);
cudaError_t launch_export_phi(const double* PhiT, long n_rows, int width, int kb, const int* fmap, double* out, cudaStream_t st);
// p_acc >= 0: ratio + accept/reject + commit of electron p_acc (spin-local index); p_prop >= 0: proposal of p_prop
cudaError_t launch_step(const SysDev& s, const WalkDev& wd, int spin, int p_acc, int p_prop, long log_off, uint32_t step, double tau,
                        int commit, cudaStream_t st);
cudaError_t launch_flush(const SysDev& s, const WalkDev& wd, int spin, cudaStream_t st, int max_m = 1 << 30);   // max_m: the most moves that can be pending (delay_k): short windows flush in one kernel
cudaError_t launch_window_reset(const WalkDev& wd, cudaStream_t st);
cudaError_t launch_eloc(const SysDev& s, const WalkDev& wd, cudaStream_t st);
cudaError_t launch_gather_rp(const WalkDev& wd, int e, cudaStream_t st);
cudaError_t launch_store_init_rows(const SysDev& s, const WalkDev& wd, int spin, int p, cudaStream_t st);
// in-place inverse of the leading n x n blocks; tmp (batch * stride doubles, may be NULL) enables the blocked DMMA path
cudaError_t launch_gj_inverse(double* Mall, long stride, int n, int ld, int batch, double* logdet, int* sign, int* status, double* tmp,
                              cudaStream_t st);
cudaError_t launch_refine_inverse(const SysDev& s, const WalkDev& wd, int spin, double* E, double* Z, cudaStream_t st);
cudaError_t launch_jastrow_total(const SysDev& s, const WalkDev& wd, cudaStream_t st);
cudaError_t launch_import_positions(const WalkDev& wd, const double* in, cudaStream_t st);
cudaError_t launch_export_positions(const WalkDev& wd, double* out, cudaStream_t st);
cudaError_t launch_export_ainv(const double* AinvT, int W, int ns, int nsp, double* out, cudaStream_t st);
cudaError_t launch_export_rows(const double* src, long n_rows, int width, long ld, double* out, cudaStream_t st);
cudaError_t launch_sign_to_i8(const int* in, int n, int8_t* out, cudaStream_t st);
cudaError_t launch_fill_int(int* p, int n, int v, cudaStream_t st);
cudaError_t launch_enn(const SysDev& s, double* out, cudaStream_t st);
cudaError_t launch_dmma_peak(double* out, int grid, int threads, int iters, cudaStream_t st);
cudaError_t launch_fill_double(double* p, int n, double v, cudaStream_t st);
cudaError_t launch_dmc_begin(const WalkDev& wd, cudaStream_t st);
cudaError_t launch_dmc_weight(const WalkDev& wd, double tau, double e_trial, const double* e_trial_dev, cudaStream_t st);
cudaError_t launch_branch(const SysDev& s, const WalkDev& wd, int* ibuf, double* e_mixed, uint32_t step, double* e_trial_dev, double feedback,
                          double* branch_log, cudaStream_t st);
bool small_path_ok(const SysDev& s, const WalkDev& wd);
// the mid-size path (window_kernel.cuh): electrons p_first .. p_first + n_steps - 1 of one spin in one launch
bool window_path_ok(const SysDev& s, const WalkDev& wd, int kp);
cudaError_t launch_window(const SysDev& s, const WalkDev& wd, int spin, int p_first, int n_steps, long log_base, int W_total, uint32_t step,
                          double tau, cudaStream_t st);
cudaError_t launch_sweep_small(const SysDev& s, const WalkDev& wd, int nsteps, uint32_t step0, double tau, int dmc, double e_trial,
                               const double* e_trial_dev, cudaStream_t st);
cudaError_t launch_plain_C(const double* in, int nb, int ns, double* Cp, int nsp, const int* fmap, cudaStream_t st);
// row f2 (first half): acc[W][n_atoms][3] += spin sp's part of d ln|Psi|/dR_a (+ the Jastrow part with spin 0); Mt: scratch [W][nsp][nbp]
cudaError_t launch_nl_count(const SysDev& s, const WalkDev& wd, const NlArgs& a, cudaStream_t st);
cudaError_t launch_nl_evaluate(const SysDev& s, const WalkDev& wd, const NlArgs& a, int n_pairs, int n_sm, unsigned* mo_epoch, double* vnl,
                               cudaStream_t st);
cudaError_t launch_forces(const SysDev& s, const WalkDev& wd, double* Mt, double* Nt, double* Bm, double* U, double* XT, double* fg,
                          double* acc_E, double* acc_psi, cudaStream_t st);
cudaError_t launch_dlogpsi_dR(const SysDev& s, const WalkDev& wd, int spin, double* Mt, double* acc, cudaStream_t st);
cudaError_t launch_philox_words(int n, const uint32_t* in, uint32_t* out, cudaStream_t st);
uint64_t launch_count();

}  // namespace qmc
