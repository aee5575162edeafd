// qmc_api.cu -- the C ABI of include/qmc.h: argument checking, device memory, and the host-side
// scheduler that enqueues the per-electron kernels of a sweep (no host synchronisation inside a sweep).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <string>
#include <vector>

#include "../../include/qmc.h"
#include "qmc_kernels.cuh"

using namespace qmc;

static constexpr size_t MO_TRACE_SLOTS = 8192;
#ifndef QMC_LANE_FREE_SMS
#define QMC_LANE_FREE_SMS 16
#endif

static thread_local std::string g_err;

static int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
#define CU(call)                                                                                            \
    do {                                                                                                    \
        cudaError_t _e = (call);                                                                            \
        if (_e != cudaSuccess) {                                                                            \
            cudaGetLastError();                                                                             \
            return fail(_e == cudaErrorMemoryAllocation ? QMC_ERR_NOMEM : QMC_ERR_CUDA,                     \
                        std::string(#call) + ": " + cudaGetErrorString(_e) + " (" __FILE__ ":" + std::to_string(__LINE__) + ")"); \
        }                                                                                                   \
    } while (0)

static inline int round_up(int x, int m) { return (x + m - 1) / m * m; }
static bool is_device_ptr(const void* p);

struct DevPool {  // owns cudaMalloc'ed blocks
    std::vector<void*> blocks;
    cudaError_t alloc(void** p, size_t bytes, cudaStream_t st, bool zero = true) {
        *p = nullptr;
        if (bytes == 0) bytes = 16;
        cudaError_t e = cudaMalloc(p, bytes);
        if (e != cudaSuccess) return e;
        blocks.push_back(*p);
        if (zero) e = cudaMemsetAsync(*p, 0, bytes, st);
        return e;
    }
    void release(void* p) {
        for (auto& b : blocks)
            if (b == p) { cudaFree(b); b = nullptr; }
    }
    void free_all() {
        for (void* b : blocks)
            if (b) cudaFree(b);
        blocks.clear();
    }
};

// A buffer that grows on demand and is kept: the scratch of the row-f2 / f3 getters and the staging buffer of the
// host-pointer getters are allocated by the first call that needs them, not by every call.
struct GrowBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes, cudaStream_t st) {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaError_t es = cudaStreamSynchronize(st); if (es != cudaSuccess) return es; cudaFree(p); p = nullptr; cap = 0; }
        cudaError_t e = cudaMalloc(&p, bytes + 256);
        if (e != cudaSuccess) { p = nullptr; return e; }
        cap = bytes;
        return cudaSuccess;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

struct qmc_system {
    SysDev d;
    DevPool pool;
    cudaStream_t stream;
    int device;
    int n_sm;
};

// Every entry point that takes a system or a walker set runs on the device the system was built on, whatever the calling
// thread's current device is; the caller's device is restored on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) { err = cudaSetDevice(device); switched = err == cudaSuccess; }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
// A non-sticky CUDA error that some earlier runtime call on this host thread left behind (ours are all checked where they
// are made; PyTorch and other libraries share the thread) would otherwise be picked up by the cudaGetLastError() that
// follows our next kernel launch and be reported as that launch's failure.  Entry points drop it and remember what it was
// (qmc_stale_error), so that it is neither mistaken for ours nor lost.
static thread_local std::string g_stale;
static void drop_stale_error(const char* where) {
    const cudaError_t se = cudaGetLastError();
    if (se != cudaSuccess) g_stale = std::string(cudaGetErrorString(se)) + " (found pending at " + where + ")";
}
extern "C" const char* qmc_stale_error(void) { return g_stale.c_str(); }
#define GUARD(sysptr)                                                                                    \
    drop_stale_error(__func__);                                                                          \
    DeviceGuard _guard((sysptr)->device);                                                                \
    if (_guard.err != cudaSuccess) { cudaGetLastError(); return fail(QMC_ERR_CUDA, std::string("cannot select the system's device: ") + cudaGetErrorString(_guard.err)); }

struct StageTimer {
    std::vector<cudaEvent_t> ev;  // pairs
    std::vector<int> stage;
    size_t used = 0;
};

// One lane of a crowd: a contiguous range of its walkers that moves through the electron steps on its own stream.  A
// large crowd runs as TWO lanes, because inside one lane an electron step is a dependency chain (basis -> contraction ->
// accept/propose) that leaves the tensor pipe idle a fifth of the time; the other lane's contraction fills those gaps, and
// this lane's HBM-bound kernels run in the shadow of it (they are sized to fit on an SM beside the resident contraction
// CTA).  Lanes share the crowd's per-walker arrays (views at an offset); each owns what one contraction needs privately.
struct Lane {
    WalkDev d;            // view of walkers [off, off + d.W)
    int off;
    cudaStream_t stream;  // lane 0: the crowd's stream
    unsigned own_epoch;   // stream-K launch counter of a private flags buffer (lane 1); lane 0 stamps the crowd's flags
    unsigned* mo_epoch;   //   buffer and therefore counts with the crowd's counter
    cudaEvent_t done;
};

struct qmc_walkers {
    const qmc_system* sys;
    WalkDev d;
    int n_lanes;
    Lane lane[2];
    cudaEvent_t fork_ev;
    DevPool pool;
    DevPool winpool;
    DevPool logpool;
    cudaStream_t stream;
    uint32_t step;       // global sweep counter (A12)
    uint32_t flags;
    int T_last;          // sweeps in the most recent qmc_sweep call
    size_t log_capacity; // entries the log buffers can hold
    int* d_status;
    int* d_comb;        // [4 W + 1] reconfiguration scratch: source, pair_dst, pair_src, mult, n_pairs
    double* d_emixed;   // [1]
    unsigned mo_epoch;   // stream-K launch counter (flag stamps)
    int prof_stride;     // 0 = off
    GrowBuf mo_trace;         // [MO_TRACE_SLOTS][n_sm][2] globaltimer stamps of the profiled contraction launches
    std::vector<int> trace_grid;  // grid of every traced launch
    mutable GrowBuf scratch;  // qmc_get_dlogpsi_dR / qmc_get_deloc_dR / qmc_get_vnl
    mutable GrowBuf bounce;   // device staging of the getters that write to host memory
    StageTimer timer;
    double stage_ms[8];
    uint64_t stage_n[8];
};

extern "C" const char* qmc_last_error(void) { return g_err.c_str(); }
extern "C" const char* qmc_version(void) { return "paper_2504_07948_b200 r2 (sm_100a, FP64 DMMA)"; }
extern "C" uint64_t qmc_launch_count(void) { return launch_count(); }

static int check_device() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(QMC_ERR_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(e)); }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(QMC_ERR_CUDA, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e)); }
    if (prop.major != 10) return fail(QMC_ERR_CUDA, "this library is built for sm_100a only (found sm_" + std::to_string(prop.major) + std::to_string(prop.minor) + "); there is no fallback path");
    return QMC_OK;
}

// ------------------------------------------------------------------------------------------------ qmc_init

template <class T>
static cudaError_t fetch(std::vector<T>& dst, const T* src, size_t n) {
    dst.resize(n);
    if (n == 0) return cudaSuccess;
    return cudaMemcpy(dst.data(), src, n * sizeof(T), cudaMemcpyDefault);
}

extern "C" int qmc_init(qmc_system** out, const qmc_atoms* atoms, const qmc_basis* basis, const qmc_mo* mo,
                        const qmc_jastrow* jas, void* cuda_stream) {
    if (!out || !atoms || !basis || !mo || !jas) return fail(QMC_ERR_ARG, "qmc_init: null argument");
    *out = nullptr;
    if (atoms->n_atoms < 1 || !atoms->xyz || !atoms->Z) return fail(QMC_ERR_ARG, "qmc_init: atoms");
    if (basis->n_shells < 1 || !basis->atom || !basis->l || !basis->n_prim || !basis->prim_offset || !basis->alpha || !basis->coef || basis->n_prim_total < 1)
        return fail(QMC_ERR_ARG, "qmc_init: basis");
    if (mo->n_basis < 1 || mo->n_up < 0 || mo->n_dn < 0 || mo->n_up + mo->n_dn < 1 || (mo->n_up > 0 && !mo->C_up) || (mo->n_dn > 0 && !mo->C_dn))
        return fail(QMC_ERR_ARG, "qmc_init: mo");
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    std::vector<double> xyz, Z, alpha, coef;
    std::vector<int> sh_atom, sh_l, sh_np, sh_off;
    CU(fetch(xyz, atoms->xyz, (size_t)3 * atoms->n_atoms));
    CU(fetch(Z, atoms->Z, (size_t)atoms->n_atoms));
    CU(fetch(sh_atom, basis->atom, (size_t)basis->n_shells));
    CU(fetch(sh_l, basis->l, (size_t)basis->n_shells));
    CU(fetch(sh_np, basis->n_prim, (size_t)basis->n_shells));
    CU(fetch(sh_off, basis->prim_offset, (size_t)basis->n_shells));
    CU(fetch(alpha, basis->alpha, (size_t)basis->n_prim_total));
    CU(fetch(coef, basis->coef, (size_t)basis->n_prim_total));

    // numeric input: the basis kernel's exp is written for arguments -alpha t <= 0, and a non-finite table entry would
    // poison every walker silently
    auto all_finite = [](const std::vector<double>& v) { for (double x : v) if (!std::isfinite(x)) return false; return true; };
    if (!all_finite(xyz) || !all_finite(Z)) return fail(QMC_ERR_ARG, "qmc_init: atom coordinates and charges must be finite");
    if (!all_finite(alpha) || !all_finite(coef)) return fail(QMC_ERR_ARG, "qmc_init: exponents and coefficients must be finite");
    for (double a : alpha)
        if (a < 0.0) return fail(QMC_ERR_ARG, "qmc_init: exponents must be >= 0");
    if (!std::isfinite(jas->a_anti) || !std::isfinite(jas->a_para) || !std::isfinite(jas->b_ee) || !std::isfinite(jas->b_en))
        return fail(QMC_ERR_ARG, "qmc_init: Jastrow parameters must be finite");
    std::vector<ShellRec> recs(basis->n_shells);
    int f = 0;
    for (int i = 0; i < basis->n_shells; i++) {
        if (sh_l[i] < 0 || sh_l[i] > 2) return fail(QMC_ERR_ARG, "qmc_init: shell angular momentum must be 0, 1 or 2");
        if (sh_atom[i] < 0 || sh_atom[i] >= atoms->n_atoms) return fail(QMC_ERR_ARG, "qmc_init: shell atom index out of range");
        if (sh_np[i] < 1 || sh_off[i] < 0 || sh_off[i] + sh_np[i] > basis->n_prim_total) return fail(QMC_ERR_ARG, "qmc_init: primitive range out of bounds");
        recs[i].x = xyz[3 * sh_atom[i]]; recs[i].y = xyz[3 * sh_atom[i] + 1]; recs[i].z = xyz[3 * sh_atom[i] + 2];
        recs[i].l = sh_l[i]; recs[i].f0 = f; recs[i].nprim = sh_np[i]; recs[i].poff = sh_off[i];
        f += 2 * sh_l[i] + 1;
    }
    if (f != mo->n_basis) return fail(QMC_ERR_ARG, "qmc_init: n_basis != sum over shells of 2l+1");
    // Internal order of the basis functions (the K index of the contraction; any order gives the same sums up to rounding):
    // shells grouped by how far they reach -- sqrt(ln(1/theta) / smallest exponent) -- and, inside a group, along a Morton
    // curve through their centres, so that the 32 functions of a k-block die off together in space.  It is what makes the
    // optional screening (QMC_SCREEN_MO) effective; the caller's order is kept at the ABI (C rows in, qmc_eval_basis out).
    std::vector<int> order(basis->n_shells), fmap(mo->n_basis);
    {
        double lo3[3] = {1e300, 1e300, 1e300}, hi3[3] = {-1e300, -1e300, -1e300};
        for (const ShellRec& r : recs) {
            const double c[3] = {r.x, r.y, r.z};
            for (int q = 0; q < 3; q++) { lo3[q] = std::min(lo3[q], c[q]); hi3[q] = std::max(hi3[q], c[q]); }
        }
        std::vector<uint64_t> key(basis->n_shells);
        for (int i = 0; i < basis->n_shells; i++) {
            double amin = 1e300;
            for (int q = 0; q < recs[i].nprim; q++) amin = std::min(amin, fabs(alpha[recs[i].poff + q]));
            const double reach = amin > 0.0 ? sqrt(55.0 / amin) : 1e300;
            int cls = 0;
            for (double edge : {3.0, 5.0, 8.0, 12.0, 17.0}) cls += reach > edge;
            const double c[3] = {recs[i].x, recs[i].y, recs[i].z};
            uint64_t mort = 0;
            for (int q = 0; q < 3; q++) {
                const double span = hi3[q] - lo3[q];
                uint64_t v = span > 0.0 ? (uint64_t)((c[q] - lo3[q]) / span * 1023.0) : 0;
                for (int b = 0; b < 10; b++) mort |= ((v >> b) & 1ull) << (3 * b + q);
            }
            key[i] = ((uint64_t)cls << 32) | mort;
            order[i] = i;
        }
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key[a] < key[b]; });
        int fn = 0;
        for (int i : order) {
            for (int m = 0; m < 2 * recs[i].l + 1; m++) fmap[recs[i].f0 + m] = fn + m;
            recs[i].f0 = fn;
            fn += 2 * recs[i].l + 1;
        }
    }

    qmc_system* S = new qmc_system();
    S->stream = st;
    cudaGetDevice(&S->device);
    SysDev& d = S->d;
    memset(&d, 0, sizeof(d));
    d.n_atoms = atoms->n_atoms; d.n_shells = basis->n_shells; d.n_basis = mo->n_basis; d.nbp = round_up(mo->n_basis, 32); d.kb = d.nbp / 32;
    d.ns[0] = mo->n_up; d.ns[1] = mo->n_dn; d.nsp[0] = round_up(mo->n_up, 16); d.nsp[1] = round_up(mo->n_dn, 16);
    d.nt[0] = (d.nsp[0] + 127) / 128; d.nt[1] = (d.nsp[1] + 127) / 128;
    d.ne = mo->n_up + mo->n_dn;
    cudaDeviceGetAttribute(&S->n_sm, cudaDevAttrMultiProcessorCount, S->device);
    d.a_anti = jas->a_anti; d.a_para = jas->a_para; d.b_ee = jas->b_ee; d.b_en = jas->b_en;
    auto cleanup = [&](int code, const std::string& m) { S->pool.free_all(); delete S; return fail(code, m); };
#define CUS(call)                                                                                       \
    do {                                                                                                \
        cudaError_t _e = (call);                                                                        \
        if (_e != cudaSuccess) { cudaGetLastError(); return cleanup(_e == cudaErrorMemoryAllocation ? QMC_ERR_NOMEM : QMC_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(_e)); } \
    } while (0)
    double *dxyz, *dZ, *dal, *dco, *denn;
    ShellRec* drec;
    CUS(S->pool.alloc((void**)&dxyz, xyz.size() * 8, st));
    CUS(S->pool.alloc((void**)&dZ, Z.size() * 8, st));
    CUS(S->pool.alloc((void**)&dal, alpha.size() * 8, st));
    CUS(S->pool.alloc((void**)&dco, coef.size() * 8, st));
    CUS(S->pool.alloc((void**)&drec, recs.size() * sizeof(ShellRec), st));
    CUS(S->pool.alloc((void**)&denn, 8, st));
    CUS(cudaMemcpyAsync(dxyz, xyz.data(), xyz.size() * 8, cudaMemcpyHostToDevice, st));
    CUS(cudaMemcpyAsync(dZ, Z.data(), Z.size() * 8, cudaMemcpyHostToDevice, st));
    CUS(cudaMemcpyAsync(dal, alpha.data(), alpha.size() * 8, cudaMemcpyHostToDevice, st));
    CUS(cudaMemcpyAsync(dco, coef.data(), coef.size() * 8, cudaMemcpyHostToDevice, st));
    CUS(cudaMemcpyAsync(drec, recs.data(), recs.size() * sizeof(ShellRec), cudaMemcpyHostToDevice, st));
    d.atom_xyz = dxyz; d.atom_Z = dZ; d.alpha = dal; d.coef = dco; d.shells = drec;
    {   // shells that own a function of each 32-function k-block (a shell may straddle two blocks), grouped by l
        std::vector<int4> cnts(d.kb);
        std::vector<KbShell> list;
        int lo = 0;  // positions in `order` (the shells sorted by their first internal function)
        for (int kb = 0; kb < d.kb; kb++) {
            const int f_lo = kb * 32, f_hi = f_lo + 32;
            while (lo < basis->n_shells && recs[order[lo]].f0 + 2 * recs[order[lo]].l + 1 <= f_lo) lo++;
            int hi = lo;
            while (hi < basis->n_shells && recs[order[hi]].f0 < f_hi) hi++;
            int c[3] = {0, 0, 0};
            const int off = (int)list.size();
            for (int l = 0; l < 3; l++)
                for (int oi = lo; oi < hi; oi++)
                    if (const int i = order[oi]; recs[i].l == l) {
                        KbShell k;
                        memset(&k, 0, sizeof(k));
                        k.x = recs[i].x; k.y = recs[i].y; k.z = recs[i].z;
                        k.l = recs[i].l; k.f0 = recs[i].f0; k.nprim = recs[i].nprim; k.poff = recs[i].poff;
                        for (int q = 0; q < 3 && q < recs[i].nprim; q++) { k.a[q] = alpha[recs[i].poff + q]; k.c[q] = coef[recs[i].poff + q]; }
                        list.push_back(k);
                        c[l]++;
                    }
            cnts[kb] = make_int4(c[0], c[1], c[2], off);
            KbShell zero;
            memset(&zero, 0, sizeof(zero));
            list.resize(off + 32, zero);  // fixed 32 slots per block (a block of 32 functions has at most 32 shells)
        }
        if (list.empty()) { KbShell k; memset(&k, 0, sizeof(k)); list.push_back(k); }
        int4* dcn;
        KbShell* dli;
        CUS(S->pool.alloc((void**)&dcn, cnts.size() * sizeof(int4), st));
        CUS(S->pool.alloc((void**)&dli, list.size() * sizeof(KbShell), st));
        CUS(cudaMemcpyAsync(dcn, cnts.data(), cnts.size() * sizeof(int4), cudaMemcpyHostToDevice, st));
        CUS(cudaMemcpyAsync(dli, list.data(), list.size() * sizeof(KbShell), cudaMemcpyHostToDevice, st));
        CUS(cudaStreamSynchronize(st));
        d.kb_counts = dcn;
        d.kb_list = dli;
        {   // occupied slots for the window kernel: first the k-blocks of the lower half of K, each half ordered by l
            std::vector<int> items;
            const int kbh = (d.kb + 1) / 2;
            for (int half = 0; half < 2; half++) {
                for (int l = 0; l < 3; l++)
                    for (int kb = half ? kbh : 0; kb < (half ? d.kb : kbh); kb++) {
                        const int c[3] = {cnts[kb].x, cnts[kb].y, cnts[kb].z};
                        int first = 0;
                        for (int q = 0; q < l; q++) first += c[q];
                        for (int q = 0; q < c[l]; q++) items.push_back(kb * 32 + first + q);
                    }
                if (half == 0) d.n_win_first = (int)items.size();
            }
            d.n_win_items = (int)items.size();
            if (items.empty()) items.push_back(0);
            int* dwi;
            CUS(S->pool.alloc((void**)&dwi, items.size() * sizeof(int), st));
            CUS(cudaMemcpyAsync(dwi, items.data(), items.size() * sizeof(int), cudaMemcpyHostToDevice, st));
            CUS(cudaStreamSynchronize(st));
            d.win_items = dwi;
        }
        int* dfm;
        CUS(S->pool.alloc((void**)&dfm, fmap.size() * sizeof(int), st));
        CUS(cudaMemcpyAsync(dfm, fmap.data(), fmap.size() * sizeof(int), cudaMemcpyHostToDevice, st));
        CUS(cudaStreamSynchronize(st));
        d.fmap = dfm;
        // shells grouped by atom (row f2: d ln|Psi| / d R_a)
        std::vector<int> aoff(atoms->n_atoms + 1, 0), alist(basis->n_shells);
        for (int i = 0; i < basis->n_shells; i++) aoff[sh_atom[i] + 1]++;
        for (int a = 0; a < atoms->n_atoms; a++) aoff[a + 1] += aoff[a];
        {
            std::vector<int> fill(aoff.begin(), aoff.end() - 1);
            for (int i = 0; i < basis->n_shells; i++) alist[fill[sh_atom[i]]++] = i;
        }
        int *daoff, *dalist;
        CUS(S->pool.alloc((void**)&daoff, aoff.size() * sizeof(int), st));
        CUS(S->pool.alloc((void**)&dalist, alist.size() * sizeof(int) + 4, st));
        CUS(cudaMemcpyAsync(daoff, aoff.data(), aoff.size() * sizeof(int), cudaMemcpyHostToDevice, st));
        CUS(cudaMemcpyAsync(dalist, alist.data(), alist.size() * sizeof(int), cudaMemcpyHostToDevice, st));
        CUS(cudaStreamSynchronize(st));
        d.atom_shell_off = daoff;
        d.atom_shell_list = dalist;
    }
    for (int sp = 0; sp < 2; sp++) {
        double* dC;
        CUS(S->pool.alloc((void**)&dC, (size_t)d.nt[sp] * d.kb * 32 * 132 * 8, st));
        d.CT[sp] = dC;
        const double* src = sp == 0 ? mo->C_up : mo->C_dn;
        if (d.ns[sp] > 0) {
            double* tmp;  // stage (host or device source) -> device, then tile on the device
            size_t bytes = (size_t)d.n_basis * d.ns[sp] * 8;
            CUS(cudaMalloc((void**)&tmp, bytes));
            cudaError_t e = cudaMemcpyAsync(tmp, src, bytes, cudaMemcpyDefault, st);
            double* dCp = nullptr;  // plain copy in the internal function order, zero-padded to [nbp][nsp]
            if (e == cudaSuccess) e = S->pool.alloc((void**)&dCp, (size_t)d.nbp * d.nsp[sp] * 8, st);
            d.Cplain[sp] = dCp;
            if (e == cudaSuccess) e = launch_tile_C(tmp, d.n_basis, d.ns[sp], dC, d.kb, d.fmap, st);
            if (e == cudaSuccess) e = launch_plain_C(tmp, d.n_basis, d.ns[sp], dCp, d.nsp[sp], d.fmap, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            cudaFree(tmp);
            CUS(e);
        }
    }
    CUS(launch_enn(d, denn, st));
    CUS(cudaMemcpyAsync(&d.e_nn, denn, 8, cudaMemcpyDeviceToHost, st));
    CUS(cudaStreamSynchronize(st));
    *out = S;
    return QMC_OK;
}

extern "C" void qmc_finalize(qmc_system* sys) {
    if (!sys) return;
    DeviceGuard guard(sys->device);
    sys->pool.free_all();
    delete sys;
}

// ------------------------------------------------------------------------------------------------ walkers

static int alloc_window(qmc_walkers* w, int kp) {
    WalkDev& d = w->d;
    const SysDev& s = w->sys->d;
    cudaStream_t st = w->stream;
    CU(cudaStreamSynchronize(st));
    w->winpool.free_all();
    const int nspm = d.ldv;
    d.kp = kp;
    CU(w->winpool.alloc((void**)&d.Vbuf, (size_t)d.W * kp * nspm * 8, st));
    CU(w->winpool.alloc((void**)&d.Wbuf, (size_t)d.W * kp * nspm * 8, st));
    CU(w->winpool.alloc((void**)&d.W2, (size_t)d.W * kp * nspm * 8, st));
    CU(w->winpool.alloc((void**)&d.SinvT, (size_t)d.W * kp * kp * 8, st));
    CU(w->winpool.alloc((void**)&d.YT, (size_t)d.W * nspm * kp * 8, st));
    CU(w->winpool.alloc((void**)&d.bvec, (size_t)d.W * kp * 8, st));
    CU(w->winpool.alloc((void**)&d.cvec, (size_t)d.W * kp * 8, st));
    CU(w->winpool.alloc((void**)&d.plist, (size_t)d.W * kp * 4, st));
    (void)s;
    return QMC_OK;
}

static void destroy_walkers(qmc_walkers* w) {
    if (!w) return;
    cudaStreamSynchronize(w->stream);
    for (cudaEvent_t e : w->timer.ev) cudaEventDestroy(e);
    if (w->n_lanes == 2) {
        cudaStreamSynchronize(w->lane[1].stream);
        cudaStreamDestroy(w->lane[1].stream);
        cudaEventDestroy(w->lane[0].done);
        cudaEventDestroy(w->lane[1].done);
        cudaEventDestroy(w->fork_ev);
    }
    w->scratch.release();
    w->bounce.release();
    w->mo_trace.release();
    w->pool.free_all();
    w->winpool.free_all();
    w->logpool.free_all();
    delete w;
}

// 64-row units of contraction work for `rows` rows, mirroring launch_mo's choice of tile height
static int mo_row_units(const SysDev& s, int spin, int rows, int grid) {
    const int mt = (rows + 127) / 128;
    const bool half = (long)mt * s.nt[spin] * s.kb < 16L * grid || mt * 128 - rows >= 64;
    return half ? (rows + 63) / 64 : 2 * mt;
}

// Two lanes where it pays: the per-electron kernels (not the one-launch path), rows long enough for the 256-thread step
// kernel, and a crowd that splits without adding more than 5 % of padded rows to the contraction (config 2: 1280 rows = 10
// tiles -> 5 + 5; config 3: 320 rows = five 64-row tiles -> 3 + 3, so it stays one lane).
static int choose_lanes(const qmc_system* sys, const WalkDev& d, uint32_t flags) {
    const SysDev& s = sys->d;
    if ((flags & QMC_ONE_LANE) || d.W < 2) return 1;
    if (!(flags & QMC_LARGE_PATH) && small_path_ok(s, d)) return 1;
    const int nspm = s.nsp[0] > s.nsp[1] ? s.nsp[0] : s.nsp[1];
    if (nspm <= 256) return 1;
    const int w0 = (d.W + 1) / 2, w1 = d.W - w0;
    for (int sp = 0; sp < 2; sp++) {
        if (s.ns[sp] == 0) continue;
        const int whole = mo_row_units(s, sp, 5 * d.W, sys->n_sm);
        const int split = mo_row_units(s, sp, 5 * w0, sys->n_sm) + mo_row_units(s, sp, 5 * w1, sys->n_sm);
        if (split * 100 > whole * 105) return 1;
    }
    return 2;
}

// (re)build the lane views from the crowd's arrays -- after creation and whenever the delay window was re-allocated
static void build_lane_views(qmc_walkers* w) {
    const SysDev& s = w->sys->d;
    const WalkDev& d = w->d;
    const int w0 = w->n_lanes == 2 ? (d.W + 1) / 2 : d.W;
    for (int l = 0; l < w->n_lanes; l++) {
        Lane& L = w->lane[l];
        WalkDev own = L.d;  // the lane's private buffers survive the rebuild
        L.off = l == 0 ? 0 : w0;
        const long o = L.off;
        L.d = d;
        L.d.W = l == 0 ? w0 : d.W - w0;
        L.d.lean = w->n_lanes == 2 ? 1 : 0;
        L.d.R = d.R + o * 3 * d.nep;
        for (int sp = 0; sp < 2; sp++) {
            L.d.AinvT[sp] = d.AinvT[sp] + o * s.nsp[sp] * s.nsp[sp];
            L.d.Orb[sp] = d.Orb[sp] + o * 5 * s.nsp[sp] * s.nsp[sp];
        }
        L.d.V = d.V + o * 5 * d.ldv;
        L.d.Vbuf = d.Vbuf + o * d.kp * d.ldv; L.d.Wbuf = d.Wbuf + o * d.kp * d.ldv; L.d.W2 = d.W2 + o * d.kp * d.ldv;
        L.d.SinvT = d.SinvT + o * d.kp * d.kp; L.d.YT = d.YT + o * d.ldv * d.kp;
        L.d.bvec = d.bvec + o * d.kp; L.d.cvec = d.cvec + o * d.kp; L.d.xcol = d.xcol + o * d.ldv;
        L.d.plist = d.plist + o * d.kp; L.d.mcount = d.mcount + o;
        L.d.rp = d.rp + o * 3; L.d.G = d.G + o * 3; L.d.gJn = d.gJn + o * 3; L.d.u = d.u + o; L.d.dJ = d.dJ + o;
        L.d.logpsi = d.logpsi + o; L.d.sign = d.sign + o; L.d.flags = d.flags + o;
        L.d.eloc = d.eloc + o; L.d.ekin = d.ekin + o; L.d.ebuf = d.ebuf + o * s.ne * 2;
        L.d.bits = d.bits ? d.bits + o : nullptr;                       // log rows keep the crowd's stride (log_off)
        L.d.ratio_log = d.ratio_log ? d.ratio_log + o : nullptr; L.d.pacc_log = d.pacc_log ? d.pacc_log + o : nullptr;
        L.d.first_walker = d.first_walker + (uint32_t)o;
        L.d.weight = d.weight + o; L.d.eold = d.eold + o; L.d.tau_eff = d.tau_eff + o; L.d.dr2p = d.dr2p + o; L.d.dr2 = d.dr2 + o * 2;
        if (l == 1) {  // private: basis matrix, stream-K workspace and flags, screening plan
            L.d.Phi = own.Phi; L.d.mo_ws = own.mo_ws; L.d.mo_flags = own.mo_flags;
            L.d.tilemax = own.tilemax; L.d.plan_cnt = own.plan_cnt; L.d.plan_pre = own.plan_pre; L.d.plan_kb = own.plan_kb;
        }
        L.d.mt = (5 * L.d.W + 127) / 128;
    }
}

extern "C" void qmc_walkers_destroy(qmc_walkers* w) {
    if (!w) return;
    DeviceGuard guard(w->sys->device);
    destroy_walkers(w);
}

extern "C" int qmc_walkers_create(const qmc_system* sys, qmc_walkers** out, int n_walkers, const double* positions,
                                  uint64_t seed, uint32_t first_walker_id, uint32_t first_step, uint32_t flags,
                                  void* cuda_stream) {
    if (!sys || !out || !positions) return fail(QMC_ERR_ARG, "qmc_walkers_create: null argument");
    GUARD(sys);
    *out = nullptr;
    if (n_walkers < 1) return fail(QMC_ERR_ARG, "qmc_walkers_create: n_walkers < 1");
    int rc = check_device();
    if (rc) return rc;
    const SysDev& s = sys->d;
    qmc_walkers* w = new qmc_walkers();
    w->sys = sys;
    w->stream = (cudaStream_t)cuda_stream;
    w->step = first_step;
    w->flags = flags;
    w->T_last = 0;
    w->log_capacity = 0;
    w->prof_stride = 0;
    memset(w->stage_ms, 0, sizeof(w->stage_ms));
    memset(w->stage_n, 0, sizeof(w->stage_n));
    cudaStream_t st = w->stream;
    WalkDev& d = w->d;
    memset(&d, 0, sizeof(d));
    d.W = n_walkers; d.ne = s.ne; d.nep = round_up(s.ne, 8);
    d.ldv = s.nsp[0] > s.nsp[1] ? s.nsp[0] : s.nsp[1];
    d.seed = seed; d.first_walker = first_walker_id;
    const size_t W = n_walkers;
#define CUW(call)                                                                                      \
    do {                                                                                               \
        cudaError_t _e = (call);                                                                       \
        if (_e != cudaSuccess) {                                                                       \
            cudaGetLastError();                                                                        \
            std::string m = std::string(#call) + ": " + cudaGetErrorString(_e);                        \
            destroy_walkers(w);                                                                        \
            return fail(_e == cudaErrorMemoryAllocation ? QMC_ERR_NOMEM : QMC_ERR_CUDA, m);            \
        }                                                                                              \
    } while (0)
    CUW(w->pool.alloc((void**)&d.R, W * 3 * d.nep * 8, st));
    for (int sp = 0; sp < 2; sp++) {
        CUW(w->pool.alloc((void**)&d.AinvT[sp], W * s.nsp[sp] * s.nsp[sp] * 8, st));
        CUW(w->pool.alloc((void**)&d.Orb[sp], W * s.nsp[sp] * 5 * s.nsp[sp] * 8, st));
    }
    d.mt = (5 * n_walkers + 127) / 128;
    CUW(w->pool.alloc((void**)&d.Phi, phiT_bytes(s, 5 * n_walkers), st));
    d.mo_grid = sys->n_sm;
    CUW(w->pool.alloc((void**)&d.mo_ws, mo_ws_bytes(sys->n_sm), st));
    CUW(w->pool.alloc((void**)&d.mo_flags, (size_t)sys->n_sm * 4, st));
    w->mo_epoch = 0;
    CUW(w->pool.alloc((void**)&d.V, W * 5 * d.ldv * 8, st));
    CUW(w->pool.alloc((void**)&d.xcol, W * d.ldv * 8, st));
    CUW(w->pool.alloc((void**)&d.mcount, W * 4, st));
    CUW(w->pool.alloc((void**)&d.rp, W * 3 * 8, st));
    CUW(w->pool.alloc((void**)&d.G, W * 3 * 8, st));
    CUW(w->pool.alloc((void**)&d.u, W * 8, st));
    CUW(w->pool.alloc((void**)&d.dJ, W * 8, st));
    CUW(w->pool.alloc((void**)&d.gJn, W * 3 * 8, st));
    CUW(w->pool.alloc((void**)&d.logpsi, W * 8, st));
    CUW(w->pool.alloc((void**)&d.sign, W * 4, st));
    CUW(w->pool.alloc((void**)&d.flags, W * 4, st));
    CUW(w->pool.alloc((void**)&d.eloc, W * 8, st));
    CUW(w->pool.alloc((void**)&d.ekin, W * 8, st));
    CUW(w->pool.alloc((void**)&d.ebuf, W * s.ne * 2 * 8, st));
    CUW(w->pool.alloc((void**)&d.stats, 4 * 8, st));
    CUW(w->pool.alloc((void**)&d.weight, W * 8, st));
    CUW(w->pool.alloc((void**)&d.eold, W * 8, st));
    CUW(w->pool.alloc((void**)&d.dr2, W * 2 * 8, st));
    CUW(w->pool.alloc((void**)&d.dr2p, W * 8, st));
    CUW(w->pool.alloc((void**)&d.tau_eff, W * 8, st));
    CUW(w->pool.alloc((void**)&w->d_comb, (4 * W + 1) * 4, st));
    CUW(w->pool.alloc((void**)&w->d_emixed, 8, st));
    CUW(launch_fill_double(d.weight, n_walkers, 1.0, st));
    d.onepass = (flags & QMC_STEP_ONEPASS) ? 1 : 0;
    d.screen_theta = (flags & QMC_SCREEN_MO) ? QMC_SCREEN_THETA : -1.0;
    CUW(w->pool.alloc((void**)&d.tilemax, (size_t)d.mt * s.kb * 8, st));
    CUW(w->pool.alloc((void**)&d.plan_cnt, (size_t)d.mt * 4, st));
    CUW(w->pool.alloc((void**)&d.plan_pre, (size_t)(d.mt + 1) * 4, st));
    CUW(w->pool.alloc((void**)&d.plan_kb, (size_t)d.mt * s.kb * 4, st));
    CUW(w->pool.alloc((void**)&d.mo_work, 2 * 8, st));
    CUW(w->pool.alloc((void**)&w->d_status, 4, st));
    rc = alloc_window(w, 16);
    if (rc) { std::string m = g_err; destroy_walkers(w); return fail(rc, m); }
    w->n_lanes = 1;
    memset(w->lane, 0, sizeof(w->lane));
    w->lane[0].stream = st;
    w->lane[0].mo_epoch = &w->mo_epoch;
    w->lane[1].mo_epoch = &w->lane[1].own_epoch;
    if (choose_lanes(sys, d, flags) == 2) {
        Lane& L = w->lane[1];
        const int w1 = n_walkers - (n_walkers + 1) / 2, mt1 = (5 * w1 + 127) / 128;
        CUW(cudaStreamCreateWithFlags(&L.stream, cudaStreamNonBlocking));
        CUW(cudaEventCreateWithFlags(&w->fork_ev, cudaEventDisableTiming));
        CUW(cudaEventCreateWithFlags(&w->lane[0].done, cudaEventDisableTiming));
        CUW(cudaEventCreateWithFlags(&L.done, cudaEventDisableTiming));
        w->n_lanes = 2;
        // Two lanes: each contraction leaves a few SMs to the other lane's kernels.  The step / basis CTAs that share an SM
        // with a contraction CTA run slowly (one CTA per SM, the FP64 pipe taken); the ones that find a free SM run at
        // full speed and shorten the lane's chain.  Measured at config 2 (moves/s): 148 CTAs 423 k, 140: 429 k, 132:
        // 465 k, 124: 457 k, 116: 460 k (one lane: 436 k).  qmc_set_mo_ctas overrides.
        if (sys->n_sm > 4 * QMC_LANE_FREE_SMS) d.mo_grid = sys->n_sm - QMC_LANE_FREE_SMS;
        CUW(w->pool.alloc((void**)&L.d.Phi, phiT_bytes(s, 5 * w1), st));
        CUW(w->pool.alloc((void**)&L.d.mo_ws, mo_ws_bytes(sys->n_sm), st));
        CUW(w->pool.alloc((void**)&L.d.mo_flags, (size_t)sys->n_sm * 4, st));
        CUW(w->pool.alloc((void**)&L.d.tilemax, (size_t)mt1 * s.kb * 8, st));
        CUW(w->pool.alloc((void**)&L.d.plan_cnt, (size_t)mt1 * 4, st));
        CUW(w->pool.alloc((void**)&L.d.plan_pre, (size_t)(mt1 + 1) * 4, st));
        CUW(w->pool.alloc((void**)&L.d.plan_kb, (size_t)mt1 * s.kb * 4, st));
    }

    // positions in (host or device) -> walker-major SoA
    {
        double* tmp;
        size_t bytes = W * s.ne * 3 * 8;
        CUW(cudaMalloc((void**)&tmp, bytes));
        cudaError_t e = cudaMemcpyAsync(tmp, positions, bytes, cudaMemcpyDefault, st);
        if (e == cudaSuccess) e = launch_import_positions(d, tmp, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(tmp);
        CUW(e);
    }
    CUW(launch_fill_int(d.sign, n_walkers, 1, st));
    // scratch for the blocked inversion and the Newton-Schulz step (freed before returning)
    const size_t mat_max = (size_t)d.ldv * d.ldv * 8;
    double *E = nullptr, *Z = nullptr;
    CUW(cudaMalloc((void**)&E, W * mat_max + 16));
    {
        cudaError_t ez = cudaMalloc((void**)&Z, W * mat_max + 16);
        if (ez != cudaSuccess) { cudaFree(E); CUW(ez); }
    }
#define CUF(call)                                                                                      \
    do {                                                                                               \
        const cudaError_t _ef = (call);   /* (not _e: CUW declares its own) */                       \
        if (_ef != cudaSuccess) { cudaStreamSynchronize(st); cudaFree(E); cudaFree(Z); CUW(_ef); }     \
    } while (0)
    // orbital rows of every electron: basis kernel + FP64 contraction, one electron index at a time
    for (int sp = 0; sp < 2; sp++) {
        const int e0 = sp == 0 ? 0 : s.ns[0];
        for (int p = 0; p < s.ns[sp]; p++) {
            CUF(launch_gather_rp(d, e0 + p, st));
            CUF(launch_basis(s, d.rp, n_walkers, d.Phi, nullptr, st));
            CUF(launch_mo(s, sp, d.Phi, 5 * n_walkers, d.V, d.ldv, d.mo_ws, d.mo_flags, mo_grid_for(s, sp, 5 * n_walkers, d.mo_grid), ++w->mo_epoch, nullptr, st));
            CUF(launch_store_init_rows(s, d, sp, p, st));
        }
        CUF(launch_gj_inverse(d.AinvT[sp], (long)s.nsp[sp] * s.nsp[sp], s.ns[sp], s.nsp[sp], n_walkers, d.logpsi, d.sign, w->d_status, E, st));
    }
    int status = 0;
    CUF(cudaMemcpyAsync(&status, w->d_status, 4, cudaMemcpyDeviceToHost, st));
    CUF(cudaStreamSynchronize(st));
    if (status != 0) {
        cudaFree(E);
        cudaFree(Z);
        destroy_walkers(w);
        return fail(QMC_ERR_SINGULAR, "qmc_walkers_create: singular Slater matrix (zero pivot)");
    }
    // one Newton-Schulz refinement step of every inverse
    for (int sp = 0; sp < 2; sp++) CUF(launch_refine_inverse(s, d, sp, E, Z, st));
    CUF(cudaStreamSynchronize(st));
    cudaFree(E);
    cudaFree(Z);
    CUW(launch_jastrow_total(s, d, st));
    CUW(launch_window_reset(d, st));
    CUW(launch_eloc(s, d, st));
    CUW(cudaStreamSynchronize(st));
    *out = w;
    return QMC_OK;
}

// ------------------------------------------------------------------------------------------------ profiling hooks

static void prof_begin(qmc_walkers* w, cudaStream_t stream, int stage, bool on) {
    if (!on) return;
    StageTimer& t = w->timer;
    if (t.used + 2 > t.ev.size()) {
        cudaEvent_t a, b;
        cudaEventCreate(&a);
        cudaEventCreate(&b);
        t.ev.push_back(a);
        t.ev.push_back(b);
    }
    t.stage.resize(t.ev.size() / 2);
    t.stage[t.used / 2] = stage;
    cudaEventRecord(t.ev[t.used], stream);
}
static void prof_end(qmc_walkers* w, cudaStream_t stream, bool on) {
    if (!on) return;
    StageTimer& t = w->timer;
    cudaEventRecord(t.ev[t.used + 1], stream);
    t.used += 2;
}
static void prof_collect(qmc_walkers* w) {
    StageTimer& t = w->timer;
    if (t.used == 0) return;
    cudaStreamSynchronize(w->stream);
    if (w->n_lanes == 2) cudaStreamSynchronize(w->lane[1].stream);
    for (size_t i = 0; i < t.used; i += 2) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, t.ev[i], t.ev[i + 1]) == cudaSuccess) {
            w->stage_ms[t.stage[i / 2]] += ms;
            w->stage_n[t.stage[i / 2]] += 1;
        }
    }
    t.used = 0;
}

/* stage ids: 0 step kernel with one half (first proposal / last accept of a delay window), 1 basis, 2 MO contraction,
   3 fused step kernel (accept of p + proposal of p + 1), 4 flush, 5 local energy, 6 window kernel (mid-size path: all
   electron steps of one delay window in one launch) */
extern "C" int qmc_set_profiling(qmc_walkers* w, int stride) {
    if (!w || stride < 0) return fail(QMC_ERR_ARG, "qmc_set_profiling");
    GUARD(w->sys);
    prof_collect(w);
    w->prof_stride = stride;
    memset(w->stage_ms, 0, sizeof(w->stage_ms));
    memset(w->stage_n, 0, sizeof(w->stage_n));
    w->trace_grid.clear();
    if (stride > 0) CU(w->mo_trace.reserve(MO_TRACE_SLOTS * 2 * (size_t)w->sys->n_sm * 8, w->stream));
    return QMC_OK;
}
extern "C" int qmc_get_stage_times(qmc_walkers* w, double* ms /*[7]*/, uint64_t* counts /*[7]*/) {
    if (!w || !ms || !counts) return fail(QMC_ERR_ARG, "qmc_get_stage_times");
    GUARD(w->sys);
    prof_collect(w);
    for (int i = 0; i < 7; i++) { ms[i] = w->stage_ms[i]; counts[i] = w->stage_n[i]; }
    return QMC_OK;
}

// ------------------------------------------------------------------------------------------------ qmc_sweep

// dmc != 0: every sweep is a DMC generation (row f1): limited drift, then the weight update after E_L
// e_trial_dev != nullptr: E_T is read from the device.  The accept / ratio logs of this call are steps log_t0 .. log_t0 +
// nsteps - 1 of a log of log_T steps (log_T < 0: the call is the whole log).
struct SweepCall {
    int nsteps; double tau; int delay_k; int dmc; double e_trial; double lim_a;
    const double* e_trial_dev; int log_t0; int log_T;
};

// argument checks, delay window and log buffers of one walker set; *small: the set takes the one-launch path
static int sweep_prepare(qmc_walkers* w, SweepCall& c, bool* small) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_sweep: null walkers");
    if (c.nsteps < 0) return fail(QMC_ERR_ARG, "qmc_sweep: nsteps < 0");
    if (!(c.tau > 0.0) || !isfinite(c.tau)) return fail(QMC_ERR_ARG, "qmc_sweep: tau must be > 0");
    if (c.delay_k < 1 || c.delay_k > 128) return fail(QMC_ERR_ARG, "qmc_sweep: delay_k must be in 1..128");
    if (c.dmc && (!isfinite(c.e_trial) || !(c.lim_a >= 0.0) || !isfinite(c.lim_a))) return fail(QMC_ERR_ARG, "qmc_dmc_step: e_trial must be finite and limiter_a >= 0");
    const SysDev& s = w->sys->d;
    WalkDev& d = w->d;
    cudaStream_t st = w->stream;
    d.lim_a = c.dmc ? c.lim_a : 0.0;
    const int kp = round_up(c.delay_k, 16);
    if (kp != d.kp) {
        int rc = alloc_window(w, kp);
        if (rc) return rc;
        CU(launch_window_reset(d, st));
    }
    // accept / ratio logs of this call: the buffers are kept from call to call and only grow, so that a loop of
    // qmc_sweep calls of the same length never synchronises with the host
    if (c.log_T < 0) c.log_T = c.nsteps;
    const size_t nlog = (size_t)c.log_T * s.ne * d.W;
    if (nlog > w->log_capacity || !d.bits) {
        CU(cudaStreamSynchronize(st));
        w->logpool.free_all();
        d.bits = nullptr; d.ratio_log = nullptr; d.pacc_log = nullptr;
        w->log_capacity = 0;
        CU(w->logpool.alloc((void**)&d.bits, nlog, st, false));
        if (w->flags & QMC_LOG_RATIOS) {
            CU(w->logpool.alloc((void**)&d.ratio_log, nlog * 8, st, false));
            CU(w->logpool.alloc((void**)&d.pacc_log, nlog * 8, st, false));
        }
        w->log_capacity = nlog;
    }
    w->T_last = c.log_T;
    *small = !(w->flags & QMC_LARGE_PATH) && small_path_ok(s, d);
    return QMC_OK;
}

// row f4: the whole call of one set in one launch
static int sweep_small(qmc_walkers* w, const SweepCall& c) {
    const SysDev& s = w->sys->d;
    WalkDev dl = w->d;
    const size_t off = (size_t)c.log_t0 * s.ne * dl.W;
    dl.bits += off;
    if (dl.ratio_log) { dl.ratio_log += off; dl.pacc_log += off; }
    if (c.nsteps > 0) CU(launch_sweep_small(s, dl, c.nsteps, w->step, c.tau, c.dmc, c.e_trial, c.e_trial_dev, w->stream));
    w->step += (uint32_t)c.nsteps;
    return QMC_OK;
}

// everything one lane launches for electron p of spin sp in sweep t of the call; in_window: moves pending in its delay window
static int sweep_electron(qmc_walkers* w, Lane& L, const SweepCall& c, int t, int sp, int p, int* in_window) {
    const SysDev& s = w->sys->d;
    const WalkDev& d = L.d;
    cudaStream_t st = L.stream;
    const int ns = s.ns[sp], e0 = sp == 0 ? 0 : s.ns[0];
    const int e = e0 + p;
    const long log_off = ((long)(c.log_t0 + t) * s.ne + e) * w->d.W;   // the crowd's stride: the lane's log pointers are offset
    const bool prof = w->prof_stride > 0 && (p % w->prof_stride) == 0;
    const bool pf = w->prof_stride > 0;
    if (*in_window == 0) {  // first proposal of a window: nothing to fuse it with
        prof_begin(w, st, 0, pf);
        CU(launch_step(s, d, sp, -1, p, 0, w->step, c.tau, 1, st));
        prof_end(w, st, pf);
    }
    prof_begin(w, st, 1, prof);
    const bool screen = d.screen_theta >= 0.0;
    CU(launch_basis(s, d.rp, d.W, d.Phi, screen ? d.tilemax : nullptr, st));
    prof_end(w, st, prof);
    prof_begin(w, st, 2, prof);
    if (screen) CU(launch_mo_plan(s, sp, d, 5 * d.W, st));
    const int mgrid = mo_grid_for(s, sp, 5 * d.W, w->d.mo_grid);
    unsigned long long* trace = nullptr;
    if (prof && w->mo_trace.p && w->trace_grid.size() < MO_TRACE_SLOTS) {
        trace = (unsigned long long*)w->mo_trace.p + w->trace_grid.size() * 2 * (size_t)w->sys->n_sm;
        w->trace_grid.push_back(mgrid);
    }
    CU(launch_mo(s, sp, d.Phi, 5 * d.W, d.V, d.ldv, d.mo_ws, d.mo_flags, mgrid, ++*L.mo_epoch, screen ? &d : nullptr, st, trace));
    prof_end(w, st, prof);
    ++*in_window;
    if (*in_window == c.delay_k || p == ns - 1) {
        prof_begin(w, st, 0, pf);
        CU(launch_step(s, d, sp, p, -1, log_off, w->step, c.tau, 1, st));
        prof_end(w, st, pf);
        prof_begin(w, st, 4, pf);
        CU(launch_flush(s, d, sp, st, c.delay_k));
        prof_end(w, st, pf);
        *in_window = 0;
    } else {  // accept/reject of p and proposal of p + 1 in one launch
        const bool prof2 = w->prof_stride > 0 && ((p + 1) % w->prof_stride) == 0;
        prof_begin(w, st, 3, prof2);
        CU(launch_step(s, d, sp, p, p + 1, log_off, w->step, c.tau, 1, st));
        prof_end(w, st, prof2);
    }
    return QMC_OK;
}

// end of a sweep of one set: E_L, the DMC weight (lane by lane), the sweep counter
static int sweep_finish_step(qmc_walkers* w, const SweepCall& c) {
    const bool pf = w->prof_stride > 0;
    for (int l = 0; l < w->n_lanes; l++) {
        Lane& L = w->lane[l];
        prof_begin(w, L.stream, 5, pf);
        CU(launch_eloc(w->sys->d, L.d, L.stream));
        prof_end(w, L.stream, pf);
        if (c.dmc) CU(launch_dmc_weight(L.d, c.tau, c.e_trial, c.e_trial_dev, L.stream));
    }
    w->step++;
    if (w->timer.used > 8192) prof_collect(w);
    return QMC_OK;
}

// the mid-size path: one launch per delay window (window_kernel.cuh) + the flush; the whole call of one set
static int sweep_windows(qmc_walkers* w, const SweepCall& c) {
    const SysDev& s = w->sys->d;
    build_lane_views(w);
    Lane& L = w->lane[0];
    cudaStream_t st = L.stream;
    const bool pf = w->prof_stride > 0;
    if (c.dmc) CU(launch_dmc_begin(L.d, st));
    for (int t = 0; t < c.nsteps; t++) {
        const long log_base = (long)(c.log_t0 + t) * s.ne * w->d.W;
        for (int sp = 0; sp < 2; sp++)
            for (int p0 = 0; p0 < s.ns[sp]; p0 += c.delay_k) {
                const int n = s.ns[sp] - p0 < c.delay_k ? s.ns[sp] - p0 : c.delay_k;
                prof_begin(w, st, 6, pf);
                CU(launch_window(s, L.d, sp, p0, n, log_base, w->d.W, w->step, c.tau, st));
                prof_end(w, st, pf);
                prof_begin(w, st, 4, pf);
                CU(launch_flush(s, L.d, sp, st, c.delay_k));
                prof_end(w, st, pf);
            }
        int rc = sweep_finish_step(w, c);
        if (rc) return rc;
    }
    return QMC_OK;
}

// n_sets walker sets of ONE system advance together: the host enqueues electron p of every lane of every set (each on its
// own stream) before electron p + 1 of any, so that the HBM-bound stages of one lane overlap the contraction of another
static int sweep_sets(qmc_walkers* const* sets, int n_sets, SweepCall c) {
    std::vector<qmc_walkers*> large;
    for (int i = 0; i < n_sets; i++) {
        SweepCall ci = c;
        bool small = false;
        int rc = sweep_prepare(sets[i], ci, &small);
        if (rc) return rc;
        if (i == 0) c.log_T = ci.log_T;
        if (small) { rc = sweep_small(sets[i], ci); if (rc) return rc; }
        else if (!(sets[i]->flags & QMC_PER_ELECTRON) && sets[i]->n_lanes == 1 && window_path_ok(sets[i]->sys->d, sets[i]->d, sets[i]->d.kp)) {
            if (ci.nsteps > 0) { rc = sweep_windows(sets[i], ci); if (rc) return rc; }
        } else large.push_back(sets[i]);
    }
    if (large.empty() || c.nsteps == 0) return QMC_OK;
    const SysDev& s = large[0]->sys->d;
    struct Unit { qmc_walkers* w; Lane* L; int in_window; };
    std::vector<Unit> units;
    for (qmc_walkers* w : large) {
        build_lane_views(w);
        if (w->n_lanes == 2) {  // the second lane joins the crowd's stream order here and leaves it at the end of the call
            CU(cudaEventRecord(w->fork_ev, w->stream));
            CU(cudaStreamWaitEvent(w->lane[1].stream, w->fork_ev, 0));
        }
        for (int l = 0; l < w->n_lanes; l++) {
            units.push_back(Unit{w, &w->lane[l], 0});
            if (c.dmc) CU(launch_dmc_begin(w->lane[l].d, w->lane[l].stream));
        }
    }
    for (int t = 0; t < c.nsteps; t++) {
        for (int sp = 0; sp < 2; sp++)
            for (int p = 0; p < s.ns[sp]; p++)
                for (Unit& u : units) {
                    int rc = sweep_electron(u.w, *u.L, c, t, sp, p, &u.in_window);
                    if (rc) return rc;
                }
        for (qmc_walkers* w : large) {
            int rc = sweep_finish_step(w, c);
            if (rc) return rc;
        }
    }
    for (qmc_walkers* w : large)
        if (w->n_lanes == 2) {
            CU(cudaEventRecord(w->lane[1].done, w->lane[1].stream));
            CU(cudaStreamWaitEvent(w->stream, w->lane[1].done, 0));
        }
    return QMC_OK;
}

static int sweep_impl(qmc_walkers* w, int nsteps, double tau, int delay_k, int dmc, double e_trial, double lim_a,
                      const double* e_trial_dev = nullptr, int log_t0 = 0, int log_T = -1) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_sweep: null walkers");
    GUARD(w->sys);
    return sweep_sets(&w, 1, SweepCall{nsteps, tau, delay_k, dmc, e_trial, lim_a, e_trial_dev, log_t0, log_T});
}

extern "C" int qmc_sweep_crowds(qmc_walkers* const* sets, int n_sets, int nsteps, double tau, int delay_k) {
    if (!sets || n_sets < 1) return fail(QMC_ERR_ARG, "qmc_sweep_crowds: no walker sets");
    for (int i = 0; i < n_sets; i++) {
        if (!sets[i]) return fail(QMC_ERR_ARG, "qmc_sweep_crowds: null walker set");
        if (sets[i]->sys != sets[0]->sys) return fail(QMC_ERR_ARG, "qmc_sweep_crowds: the sets must belong to one system");
        for (int j = 0; j < i; j++)
            if (sets[j] == sets[i]) return fail(QMC_ERR_ARG, "qmc_sweep_crowds: a walker set appears twice");
    }
    GUARD(sets[0]->sys);
    return sweep_sets(sets, n_sets, SweepCall{nsteps, tau, delay_k, 0, 0.0, 0.0, nullptr, 0, -1});
}

extern "C" int qmc_sweep(qmc_walkers* w, int nsteps, double tau, int delay_k) { return sweep_impl(w, nsteps, tau, delay_k, 0, 0.0, 0.0); }

extern "C" int qmc_dmc_step(qmc_walkers* w, int n_generations, double tau, int delay_k, double e_trial, double limiter_a) {
    return sweep_impl(w, n_generations, tau, delay_k, 1, e_trial, limiter_a);
}

extern "C" int qmc_branch(qmc_walkers* w, int32_t* source, double* e_mixed) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_branch: null walkers");
    GUARD(w->sys);
    cudaStream_t st = w->stream;
    CU(launch_branch(w->sys->d, w->d, w->d_comb, w->d_emixed, w->step, nullptr, 0.0, nullptr, st));
    if (source) {
        CU(cudaMemcpyAsync(source, w->d_comb, (size_t)w->d.W * 4, cudaMemcpyDefault, st));
    }
    if (e_mixed) CU(cudaMemcpyAsync(e_mixed, w->d_emixed, 8, cudaMemcpyDefault, st));
    CU(cudaStreamSynchronize(st));
    return QMC_OK;
}

extern "C" int qmc_dmc_run(qmc_walkers* w, int n_generations, double tau, int delay_k, double e_trial0, double limiter_a, int branch_every,
                           double feedback, double* e_trial_out, double* branch_log, int32_t* sources) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_dmc_run: null walkers");
    GUARD(w->sys);
    if (n_generations < 0 || branch_every < 0) return fail(QMC_ERR_ARG, "qmc_dmc_run: n_generations and branch_every must be >= 0");
    if (!isfinite(e_trial0) || !isfinite(feedback)) return fail(QMC_ERR_ARG, "qmc_dmc_run: e_trial0 and feedback must be finite");
    cudaStream_t st = w->stream;
    const int W = w->d.W;
    const int n_branch = branch_every > 0 ? n_generations / branch_every : 0;
    // device side of the run: E_T, the log of the reconfigurations, their slot maps
    double* dbuf = nullptr;
    int* dsrc = nullptr;
    CU(cudaMalloc((void**)&dbuf, (size_t)(1 + 3 * (n_branch > 0 ? n_branch : 1)) * 8));
    if (sources && n_branch > 0) {
        cudaError_t e = cudaMalloc((void**)&dsrc, (size_t)n_branch * W * 4);
        if (e != cudaSuccess) { cudaFree(dbuf); CU(e); }
    }
    int rc = QMC_OK;
    cudaError_t ce = cudaMemcpyAsync(dbuf, &e_trial0, 8, cudaMemcpyHostToDevice, st);
    const int chunk = branch_every > 0 ? branch_every : (n_generations > 0 ? n_generations : 1);
    int done = 0, nb = 0;
    if (n_generations == 0 && ce == cudaSuccess) rc = sweep_impl(w, 0, tau, delay_k, 1, e_trial0, limiter_a, dbuf, 0, 0);
    while (ce == cudaSuccess && rc == QMC_OK && done < n_generations) {
        const int n = n_generations - done < chunk ? n_generations - done : chunk;
        rc = sweep_impl(w, n, tau, delay_k, 1, e_trial0, limiter_a, dbuf, done, n_generations);
        done += n;
        if (rc != QMC_OK) break;
        if (branch_every > 0 && n == chunk) {
            ce = launch_branch(w->sys->d, w->d, w->d_comb, w->d_emixed, w->step, dbuf, feedback, dbuf + 1 + 3 * nb, st);
            if (ce == cudaSuccess && dsrc) ce = cudaMemcpyAsync(dsrc + (size_t)nb * W, w->d_comb, (size_t)W * 4, cudaMemcpyDeviceToDevice, st);
            nb++;
        }
    }
    if (ce == cudaSuccess && rc == QMC_OK) {
        if (e_trial_out) ce = cudaMemcpyAsync(e_trial_out, dbuf, 8, cudaMemcpyDefault, st);
        if (ce == cudaSuccess && branch_log && n_branch > 0) ce = cudaMemcpyAsync(branch_log, dbuf + 1, (size_t)n_branch * 24, cudaMemcpyDefault, st);
        if (ce == cudaSuccess && dsrc) ce = cudaMemcpyAsync(sources, dsrc, (size_t)n_branch * W * 4, cudaMemcpyDefault, st);
    }
    cudaError_t cs = cudaStreamSynchronize(st);
    cudaFree(dbuf);
    cudaFree(dsrc);
    if (rc != QMC_OK) return rc;
    CU(ce);
    CU(cs);
    return QMC_OK;
}

extern "C" int qmc_get_dlogpsi_dR(qmc_walkers* w, double* out) {
    if (!w || !out) return fail(QMC_ERR_ARG, "qmc_get_dlogpsi_dR: null argument");
    GUARD(w->sys);
    const SysDev& s = w->sys->d;
    const WalkDev& d = w->d;
    cudaStream_t st = w->stream;
    const size_t n_out = (size_t)d.W * s.n_atoms * 3;
    const size_t n_mt = (size_t)d.W * d.ldv * s.nbp;
    if (w->scratch.reserve((n_mt + n_out + 2) * 8, st) != cudaSuccess) {
        cudaGetLastError();
        return fail(QMC_ERR_NOMEM, "qmc_get_dlogpsi_dR: scratch does not fit");
    }
    double *Mt = (double*)w->scratch.p, *acc = Mt + n_mt;
    cudaError_t e = cudaMemsetAsync(acc, 0, n_out * 8, st);
    for (int sp = 0; sp < 2 && e == cudaSuccess; sp++) e = launch_dlogpsi_dR(s, d, sp, Mt, acc, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out, acc, n_out * 8, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    CU(e);
    return QMC_OK;
}

extern "C" int qmc_get_deloc_dR(qmc_walkers* w, double* deloc, double* dlogpsi) {
    if (!w || !deloc) return fail(QMC_ERR_ARG, "qmc_get_deloc_dR: null argument");
    GUARD(w->sys);
    const SysDev& s = w->sys->d;
    const WalkDev& d = w->d;
    cudaStream_t st = w->stream;
    const size_t W = (size_t)d.W, n_out = W * s.n_atoms * 3;
    const size_t nsm = (size_t)(s.nsp[0] > s.nsp[1] ? s.nsp[0] : s.nsp[1]);
    // one allocation: Mt, Nt [W][nsm][nbp] | Bm [2][W][nsm^2] | U, XT [W][nsm^2] | fg [W][ne][8] | acc_E, acc_psi
    const size_t n_mt = W * nsm * s.nbp, n_sq = W * nsm * nsm, n_fg = W * s.ne * 8;
    const size_t total = 2 * n_mt + 4 * n_sq + n_fg + 2 * n_out + 16;
    if (w->scratch.reserve(total * 8, st) != cudaSuccess) {
        cudaGetLastError();
        return fail(QMC_ERR_NOMEM, "qmc_get_deloc_dR: scratch does not fit");
    }
    double* buf = (double*)w->scratch.p;
    double *Mt = buf, *Nt = Mt + n_mt, *Bm = Nt + n_mt, *U = Bm + 2 * n_sq, *XT = U + n_sq, *fg = XT + n_sq;
    double *accE = fg + n_fg, *accP = accE + n_out;
    cudaError_t e = cudaMemsetAsync(accE, 0, 2 * n_out * 8, st);
    if (e == cudaSuccess) e = launch_forces(s, d, Mt, Nt, Bm, U, XT, fg, accE, dlogpsi ? accP : nullptr, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(deloc, accE, n_out * 8, cudaMemcpyDefault, st);
    if (e == cudaSuccess && dlogpsi) e = cudaMemcpyAsync(dlogpsi, accP, n_out * 8, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    CU(e);
    return QMC_OK;
}

extern "C" int qmc_release_scratch(qmc_walkers* w) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_release_scratch: null walkers");
    GUARD(w->sys);
    CU(cudaStreamSynchronize(w->stream));
    w->scratch.release();
    w->bounce.release();
    return QMC_OK;
}

extern "C" int qmc_get_lanes(const qmc_walkers* w, int* n_lanes, int* walkers_per_lane) {
    if (!w || !n_lanes) return fail(QMC_ERR_ARG, "qmc_get_lanes: null argument");
    *n_lanes = w->n_lanes;
    if (walkers_per_lane) {
        const int w0 = w->n_lanes == 2 ? (w->d.W + 1) / 2 : w->d.W;
        walkers_per_lane[0] = w0;
        walkers_per_lane[1] = w->d.W - w0;
    }
    return QMC_OK;
}

extern "C" int qmc_get_mo_spans(qmc_walkers* w, double* mean_us, double* min_us, double* mean_cta_us, uint64_t* n_launches) {
    if (!w || !n_launches) return fail(QMC_ERR_ARG, "qmc_get_mo_spans: null argument");
    GUARD(w->sys);
    double mean_dummy = 0.0;
    if (!mean_us) mean_us = &mean_dummy;
    *mean_us = 0.0; *n_launches = 0;
    if (min_us) *min_us = 0.0;
    if (mean_cta_us) *mean_cta_us = 0.0;
    const size_t n = w->trace_grid.size(), nsm = (size_t)w->sys->n_sm;
    if (n == 0 || !w->mo_trace.p) return QMC_OK;
    CU(cudaStreamSynchronize(w->stream));
    if (w->n_lanes == 2) CU(cudaStreamSynchronize(w->lane[1].stream));
    std::vector<unsigned long long> h(n * 2 * nsm);
    CU(cudaMemcpy(h.data(), w->mo_trace.p, h.size() * 8, cudaMemcpyDeviceToHost));
    double sum = 0.0, mn = 1e300, sum_cta = 0.0;
    for (size_t i = 0; i < n; i++) {
        unsigned long long t0 = ~0ull, t1 = 0;
        double res = 0.0;
        for (int c = 0; c < w->trace_grid[i]; c++) {
            const unsigned long long a = h[(i * nsm + c) * 2], b = h[(i * nsm + c) * 2 + 1];
            t0 = std::min(t0, a);
            t1 = std::max(t1, b);
            res += (double)(b - a) * 1e-3;
        }
        const double us = (double)(t1 - t0) * 1e-3;
        sum += us; mn = std::min(mn, us);
        sum_cta += res / std::max(1, w->trace_grid[i]);
    }
    *mean_us = sum / n; *n_launches = n;
    if (min_us) *min_us = mn;
    if (mean_cta_us) *mean_cta_us = sum_cta / n;
    return QMC_OK;
}

extern "C" int qmc_set_ecp(qmc_system* S, int n_channels, const int32_t* ch_atom, const int32_t* ch_l, const double* ch_beta,
                           const double* ch_alpha, const double* rcut) {
    if (!S) return fail(QMC_ERR_ARG, "qmc_set_ecp: null system");
    GUARD(S);
    if (n_channels < 0 || (n_channels > 0 && (!ch_atom || !ch_l || !ch_beta || !ch_alpha)) || !rcut) return fail(QMC_ERR_ARG, "qmc_set_ecp: null argument");
    const int na = S->d.n_atoms;
    std::vector<int> atom, l;
    std::vector<double> beta, alpha, rc;
    CU(fetch(atom, ch_atom, (size_t)n_channels));
    CU(fetch(l, ch_l, (size_t)n_channels));
    CU(fetch(beta, ch_beta, (size_t)n_channels));
    CU(fetch(alpha, ch_alpha, (size_t)n_channels));
    CU(fetch(rc, rcut, (size_t)na));
    for (int c = 0; c < n_channels; c++) {
        if (atom[c] < 0 || atom[c] >= na || l[c] < 0 || l[c] > 2) return fail(QMC_ERR_ARG, "qmc_set_ecp: channel atom out of range or l not in 0..2");
        if (!isfinite(beta[c]) || !(alpha[c] >= 0.0) || !isfinite(alpha[c])) return fail(QMC_ERR_ARG, "qmc_set_ecp: beta must be finite and alpha >= 0");
    }
    for (int a = 0; a < na; a++)
        if (!(rc[a] >= 0.0) || !isfinite(rc[a])) return fail(QMC_ERR_ARG, "qmc_set_ecp: rcut must be finite and >= 0");
    // channels grouped by atom, the caller's order kept inside an atom
    std::vector<int> off(na + 1, 0), gl((size_t)n_channels);
    std::vector<double> gb((size_t)n_channels), ga((size_t)n_channels);
    for (int c = 0; c < n_channels; c++) off[atom[c] + 1]++;
    for (int a = 0; a < na; a++) off[a + 1] += off[a];
    std::vector<int> pos(off.begin(), off.end() - 1);
    for (int c = 0; c < n_channels; c++) {
        const int k = pos[atom[c]]++;
        gl[k] = l[c]; gb[k] = beta[c]; ga[k] = alpha[c];
    }
    cudaStream_t st = S->stream;
    int *d_off = nullptr, *d_l = nullptr;
    double *d_b = nullptr, *d_a = nullptr, *d_rc = nullptr;
    CU(S->pool.alloc((void**)&d_off, (size_t)(na + 1) * 4, st));
    CU(S->pool.alloc((void**)&d_l, (size_t)n_channels * 4, st));
    CU(S->pool.alloc((void**)&d_b, (size_t)n_channels * 8, st));
    CU(S->pool.alloc((void**)&d_a, (size_t)n_channels * 8, st));
    CU(S->pool.alloc((void**)&d_rc, (size_t)na * 8, st));
    CU(cudaMemcpyAsync(d_off, off.data(), (size_t)(na + 1) * 4, cudaMemcpyHostToDevice, st));
    if (n_channels > 0) {
        CU(cudaMemcpyAsync(d_l, gl.data(), (size_t)n_channels * 4, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_b, gb.data(), (size_t)n_channels * 8, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_a, ga.data(), (size_t)n_channels * 8, cudaMemcpyHostToDevice, st));
    }
    CU(cudaMemcpyAsync(d_rc, rc.data(), (size_t)na * 8, cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));
    // an earlier table stays allocated until qmc_finalize (walker sets may still be using it on their streams)
    S->d.ecp_off = d_off; S->d.ecp_l = d_l; S->d.ecp_beta = d_b; S->d.ecp_alpha = d_a; S->d.ecp_rcut = d_rc;
    return QMC_OK;
}

extern "C" int qmc_get_vnl(qmc_walkers* w, double* vnl, uint64_t* n_pairs_out) {
    if (!w || !vnl) return fail(QMC_ERR_ARG, "qmc_get_vnl: null argument");
    GUARD(w->sys);
    const SysDev& s = w->sys->d;
    const WalkDev& d = w->d;
    if (!s.ecp_off) return fail(QMC_ERR_ARG, "qmc_get_vnl: no pseudopotential set (qmc_set_ecp)");
    cudaStream_t st = w->stream;
    const size_t W = (size_t)d.W;
    // Persistent scratch (grown on demand, kept): [acc W doubles | cnt n+1 ints | per pair: 60 doubles + 3 ints].  A call
    // whose pair count exceeds what an earlier call left room for grows the buffer once; the counts are recomputed after
    // that, because growing moves the buffer.
    const size_t n_max = W * (size_t)(s.ns[0] > s.ns[1] ? s.ns[0] : s.ns[1]);
    const size_t head = ((W + 2) * 8 + (n_max + 1) * 4 + 15) / 16 * 16;
    auto pair_bytes = [](size_t np) { return np * (12 * 5 * 8 + 3 * 4) + 64; };
    cudaError_t e = w->scratch.reserve(head + pair_bytes(n_max / 2 + 1024), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(w->scratch.p, 0, W * 8, st);   // acc
    uint64_t total = 0;
    for (int sp = 0; sp < 2 && e == cudaSuccess; sp++) {
        NlArgs a;
        memset(&a, 0, sizeof(a));
        a.spin = sp; a.e0 = sp == 0 ? 0 : s.ns[0]; a.ns = s.ns[sp]; a.step = w->step;
        if (a.ns == 0) continue;
        const size_t n = W * (size_t)a.ns;
        int n_pairs = 0;
        for (int attempt = 0; attempt < 2 && e == cudaSuccess; attempt++) {
            a.cnt = (int*)((char*)w->scratch.p + (W + 2) * 8);
            e = launch_nl_count(s, d, a, st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(&n_pairs, a.cnt + n, 4, cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess || head + pair_bytes((size_t)n_pairs) <= w->scratch.cap) break;
            std::vector<double> acc_host(W);   // the sums of the spin already done move with the buffer
            e = cudaMemcpy(acc_host.data(), w->scratch.p, W * 8, cudaMemcpyDeviceToHost);
            if (e == cudaSuccess) e = w->scratch.reserve(head + pair_bytes((size_t)n_pairs), st);
            if (e == cudaSuccess) e = cudaMemcpy(w->scratch.p, acc_host.data(), W * 8, cudaMemcpyHostToDevice);
        }
        if (e == cudaSuccess && n_pairs > 0) {
            const size_t np = (size_t)n_pairs;
            double* dbuf = (double*)((char*)w->scratch.p + head);
            int* ibuf = (int*)(dbuf + np * 60);
            a.pair_w = ibuf; a.pair_e = ibuf + np; a.pair_I = ibuf + 2 * np;
            a.pts = dbuf; a.ang = dbuf + np * 36; a.terms = a.ang + np * 12;
        }
        if (e == cudaSuccess) e = launch_nl_evaluate(s, d, a, n_pairs, d.mo_grid, &w->mo_epoch, (double*)w->scratch.p, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        total += (uint64_t)n_pairs;
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(vnl, w->scratch.p, W * 8, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return fail(QMC_ERR_NOMEM, "qmc_get_vnl: scratch does not fit"); }
    CU(e);
    if (n_pairs_out) *n_pairs_out = total;
    return QMC_OK;
}

extern "C" int qmc_set_mo_ctas(qmc_walkers* w, int n_ctas) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_set_mo_ctas: null walkers");
    const int n_sm = w->sys->n_sm;
    if (n_ctas < 0 || n_ctas > n_sm) return fail(QMC_ERR_ARG, "qmc_set_mo_ctas: n_ctas must be in 0..number of SMs");
    w->d.mo_grid = n_ctas == 0 ? n_sm : n_ctas;
    return QMC_OK;
}

extern "C" int qmc_get_mo_work(const qmc_walkers* w, uint64_t* executed, uint64_t* dense) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_get_mo_work: null walkers");
    GUARD(w->sys);
    unsigned long long h[2];
    CU(cudaMemcpyAsync(h, w->d.mo_work, sizeof(h), cudaMemcpyDeviceToHost, w->stream));
    CU(cudaStreamSynchronize(w->stream));
    if (executed) *executed = h[0];
    if (dense) *dense = h[1];
    return QMC_OK;
}

extern "C" int qmc_get_weights(const qmc_walkers* w, double* weights, double* tau_eff) {
    if (!w || !weights) return fail(QMC_ERR_ARG, "qmc_get_weights: null argument");
    GUARD(w->sys);
    const size_t n = (size_t)w->d.W * 8;
    CU(cudaMemcpyAsync(weights, w->d.weight, n, cudaMemcpyDefault, w->stream));
    if (tau_eff) CU(cudaMemcpyAsync(tau_eff, w->d.tau_eff, n, cudaMemcpyDefault, w->stream));
    if (!is_device_ptr(weights) || (tau_eff && !is_device_ptr(tau_eff))) CU(cudaStreamSynchronize(w->stream));
    return QMC_OK;
}

// ------------------------------------------------------------------------------------------------ getters

static bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// run `produce(dev_buffer)` into `out` (device: directly; host: via a staging buffer + synchronous copy)
template <class F>
static int deliver(const qmc_walkers* w, void* out, size_t bytes, F&& produce) {
    cudaStream_t st = w->stream;
    if (bytes == 0) return QMC_OK;
    if (is_device_ptr(out)) {
        CU(produce(out));
        return QMC_OK;
    }
    CU(w->bounce.reserve(bytes, st));  // kept from call to call
    void* tmp = w->bounce.p;
    cudaError_t e = produce(tmp);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out, tmp, bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    CU(e);
    return QMC_OK;
}

extern "C" int qmc_get_positions(const qmc_walkers* w, double* out) {
    if (!w || !out) return fail(QMC_ERR_ARG, "qmc_get_positions: null argument");
    GUARD(w->sys);
    return deliver(w, out, (size_t)w->d.W * w->d.ne * 3 * 8, [&](void* dst) { return launch_export_positions(w->d, (double*)dst, w->stream); });
}

extern "C" int qmc_get_Ainv(const qmc_walkers* w, int spin, double* out) {
    if (!w || !out || spin < 0 || spin > 1) return fail(QMC_ERR_ARG, "qmc_get_Ainv: bad argument");
    GUARD(w->sys);
    const SysDev& s = w->sys->d;
    return deliver(w, out, (size_t)w->d.W * s.ns[spin] * s.ns[spin] * 8,
                   [&](void* dst) { return launch_export_ainv(w->d.AinvT[spin], w->d.W, s.ns[spin], s.nsp[spin], (double*)dst, w->stream); });
}

extern "C" int qmc_get_logpsi(const qmc_walkers* w, double* logabs, int8_t* sign) {
    if (!w || !logabs) return fail(QMC_ERR_ARG, "qmc_get_logpsi: null argument");
    GUARD(w->sys);
    int rc = deliver(w, logabs, (size_t)w->d.W * 8, [&](void* dst) { return cudaMemcpyAsync(dst, w->d.logpsi, (size_t)w->d.W * 8, cudaMemcpyDeviceToDevice, w->stream); });
    if (rc || !sign) return rc;
    return deliver(w, sign, (size_t)w->d.W, [&](void* dst) { return launch_sign_to_i8(w->d.sign, w->d.W, (int8_t*)dst, w->stream); });
}

extern "C" int qmc_get_eloc(const qmc_walkers* w, double* eloc, double* ekin) {
    if (!w || !eloc) return fail(QMC_ERR_ARG, "qmc_get_eloc: null argument");
    GUARD(w->sys);
    int rc = deliver(w, eloc, (size_t)w->d.W * 8, [&](void* dst) { return cudaMemcpyAsync(dst, w->d.eloc, (size_t)w->d.W * 8, cudaMemcpyDeviceToDevice, w->stream); });
    if (rc || !ekin) return rc;
    return deliver(w, ekin, (size_t)w->d.W * 8, [&](void* dst) { return cudaMemcpyAsync(dst, w->d.ekin, (size_t)w->d.W * 8, cudaMemcpyDeviceToDevice, w->stream); });
}

extern "C" int qmc_get_accept_log(const qmc_walkers* w, uint8_t* bits) {
    if (!w || !bits) return fail(QMC_ERR_ARG, "qmc_get_accept_log: null argument");
    GUARD(w->sys);
    if (!w->d.bits) return fail(QMC_ERR_STATE, "qmc_get_accept_log: no sweep has been run");
    size_t n = (size_t)w->T_last * w->d.ne * w->d.W;
    if (n == 0) return QMC_OK;
    CU(cudaMemcpyAsync(bits, w->d.bits, n, cudaMemcpyDefault, w->stream));
    if (!is_device_ptr(bits)) CU(cudaStreamSynchronize(w->stream));
    return QMC_OK;
}

extern "C" int qmc_get_ratio_log(const qmc_walkers* w, double* ratio, double* pacc) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_get_ratio_log: null walkers");
    GUARD(w->sys);
    if (!(w->flags & QMC_LOG_RATIOS) || !w->d.ratio_log) return fail(QMC_ERR_STATE, "qmc_get_ratio_log: walkers were not created with QMC_LOG_RATIOS, or no sweep has run");
    if (!ratio) return fail(QMC_ERR_ARG, "qmc_get_ratio_log: null argument");
    size_t n = (size_t)w->T_last * w->d.ne * w->d.W * 8;
    if (n == 0) return QMC_OK;
    CU(cudaMemcpyAsync(ratio, w->d.ratio_log, n, cudaMemcpyDefault, w->stream));
    if (pacc) CU(cudaMemcpyAsync(pacc, w->d.pacc_log, n, cudaMemcpyDefault, w->stream));
    if (!is_device_ptr(ratio) || (pacc && !is_device_ptr(pacc))) CU(cudaStreamSynchronize(w->stream));
    return QMC_OK;
}

extern "C" int qmc_get_stats(const qmc_walkers* w, uint64_t* n_proposed, uint64_t* n_accepted, uint64_t* n_ties, uint64_t* n_nonfinite) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_get_stats: null walkers");
    GUARD(w->sys);
    unsigned long long h[4];
    CU(cudaMemcpyAsync(h, w->d.stats, sizeof(h), cudaMemcpyDeviceToHost, w->stream));
    CU(cudaStreamSynchronize(w->stream));
    if (n_proposed) *n_proposed = h[0];
    if (n_accepted) *n_accepted = h[1];
    if (n_ties) *n_ties = h[2];
    if (n_nonfinite) *n_nonfinite = h[3];
    return QMC_OK;
}

extern "C" int qmc_synchronize(const qmc_walkers* w) {
    if (!w) return fail(QMC_ERR_ARG, "qmc_synchronize: null walkers");
    GUARD(w->sys);
    CU(cudaStreamSynchronize(w->stream));
    return QMC_OK;
}

// ------------------------------------------------------------------------------------------------ stage-level entry points

static int eval_common(const qmc_system* sys, int spin, int n_points, const double* xyz, double* out, void* cuda_stream, bool mo) {
    if (!sys || n_points < 0 || spin < 0 || spin > 1) return fail(QMC_ERR_ARG, "qmc_eval_*: bad argument");
    if (n_points == 0) return QMC_OK;
    if (!xyz || !out) return fail(QMC_ERR_ARG, "qmc_eval_*: null buffer");
    GUARD(sys);
    int rc = check_device();
    if (rc) return rc;
    const SysDev& s = sys->d;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *pts = nullptr, *Phi = nullptr, *V = nullptr, *stage = nullptr, *ws = nullptr;
    unsigned* flags = nullptr;
    const int grid = mo ? mo_grid_for(s, spin, 5 * n_points, sys->n_sm) : 0;
    const int width = mo ? s.ns[spin] : s.n_basis;
    const size_t out_bytes = (size_t)n_points * 5 * width * 8;
    cudaError_t e = cudaMalloc((void**)&pts, (size_t)n_points * 3 * 8);
    if (e == cudaSuccess) e = cudaMalloc((void**)&Phi, phiT_bytes(s, 5 * n_points));
    if (e == cudaSuccess) e = cudaMemsetAsync(Phi, 0, phiT_bytes(s, 5 * n_points), st);
    if (e == cudaSuccess && mo) e = cudaMalloc((void**)&V, (size_t)n_points * 5 * s.nsp[spin] * 8 + 16);
    if (e == cudaSuccess && mo) e = cudaMalloc((void**)&ws, mo_ws_bytes(grid) + 16);
    if (e == cudaSuccess && mo) e = cudaMalloc((void**)&flags, (size_t)grid * 4 + 16);
    if (e == cudaSuccess && mo) e = cudaMemsetAsync(flags, 0, (size_t)grid * 4 + 16, st);
    const bool dev_out = is_device_ptr(out);
    if (e == cudaSuccess && !dev_out) e = cudaMalloc((void**)&stage, out_bytes + 16);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pts, xyz, (size_t)n_points * 3 * 8, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = launch_basis(s, pts, n_points, Phi, nullptr, st);
    double* dst = dev_out ? out : stage;
    if (e == cudaSuccess) {
        if (mo) {
            e = launch_mo(s, spin, Phi, 5 * n_points, V, s.nsp[spin], ws, flags, grid, 1u, nullptr, st);
            if (e == cudaSuccess) e = launch_export_rows(V, (long)n_points * 5, width, s.nsp[spin], dst, st);
        } else {
            e = launch_export_phi(Phi, (long)n_points * 5, width, s.kb, s.fmap, dst, st);
        }
    }
    if (e == cudaSuccess && !dev_out) e = cudaMemcpyAsync(out, stage, out_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(pts); cudaFree(Phi); cudaFree(V); cudaFree(stage); cudaFree(ws); cudaFree(flags);
    CU(e);
    return QMC_OK;
}

extern "C" int qmc_eval_basis(const qmc_system* sys, int n_points, const double* xyz, double* out, void* cuda_stream) {
    return eval_common(sys, 0, n_points, xyz, out, cuda_stream, false);
}
extern "C" int qmc_eval_mo(const qmc_system* sys, int spin, int n_points, const double* xyz, double* out, void* cuda_stream) {
    return eval_common(sys, spin, n_points, xyz, out, cuda_stream, true);
}

// ---- qmc_eval_basis_noalloc: the basis kernel with its scratch (the pre-tiled A operand PhiT) in a fixed array of the
// library.  In host code `g_noalloc_scratch` is only the host-side stand-in of the symbol, never a device address: the
// address a kernel may use comes from cudaGetSymbolAddress, looked up once per device with that device current.
static __device__ __align__(256) double g_noalloc_scratch[QMC_NOALLOC_SCRATCH_BYTES / sizeof(double)];
static constexpr int NOALLOC_MAX_DEVICES = 64;
static std::atomic<double*> g_noalloc_ptr[NOALLOC_MAX_DEVICES];

static int noalloc_scratch(int device, double** out) {   // the caller has made `device` current (GUARD)
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return fail(QMC_ERR_ARG, "qmc_eval_basis_noalloc: device ordinal beyond 63");
    double* p = g_noalloc_ptr[device].load(std::memory_order_acquire);
    if (!p) {   // two threads racing here look up the same address
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(QMC_ERR_CUDA, std::string("qmc_eval_basis_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        g_noalloc_ptr[device].store(p, std::memory_order_release);
    }
    *out = p;
    return QMC_OK;
}

static bool on_device(const void* p, int device) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    if (a.type == cudaMemoryTypeManaged) return true;
    return a.type == cudaMemoryTypeDevice && a.device == device;
}

extern "C" int qmc_eval_basis_noalloc(const qmc_system* sys, int n_points, const double* xyz, double* out, void* cuda_stream) {
    if (!sys || n_points < 0) return fail(QMC_ERR_ARG, "qmc_eval_basis_noalloc: bad argument");
    if (n_points == 0) return QMC_OK;
    if (!xyz || !out) return fail(QMC_ERR_ARG, "qmc_eval_basis_noalloc: null buffer");
    GUARD(sys);
    const SysDev& s = sys->d;
    constexpr int TILE_ROWS = 128;                        // rows of one tile of PhiT (MO_BM)
    const size_t stage_bytes = phiT_bytes(s, 1);          // one tile: ceil(n_basis / 32) blocks of 128 x 36 doubles
    const long max_points = (long)(QMC_NOALLOC_SCRATCH_BYTES / stage_bytes) * TILE_ROWS / 5;
    if (n_points > max_points)
        return fail(QMC_ERR_ARG, "qmc_eval_basis_noalloc: n_points = " + std::to_string(n_points) + " needs " +
                                     std::to_string((size_t)((5L * n_points + TILE_ROWS - 1) / TILE_ROWS) * stage_bytes) + " bytes of scratch, the fixed array has " +
                                     std::to_string(QMC_NOALLOC_SCRATCH_BYTES) + ": at most " + std::to_string(max_points) +
                                     " points per call for this basis (use qmc_eval_basis, which allocates)");
    if (!on_device(xyz, sys->device) || !on_device(out, sys->device))
        return fail(QMC_ERR_ARG, "qmc_eval_basis_noalloc: xyz and out must be device memory of the system's device");
    double* PhiT = nullptr;
    int rc = noalloc_scratch(sys->device, &PhiT);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t used = phiT_bytes(s, 5 * n_points);
    // the kernel writes the real functions of the real rows only; padding must read as zero and the array keeps the last
    // call's contents
    CU(cudaMemsetAsync(PhiT, 0, used, st));
    CU(launch_basis(s, xyz, n_points, PhiT, nullptr, st));
    CU(launch_export_phi(PhiT, (long)n_points * 5, s.n_basis, s.kb, s.fmap, out, st));
    return QMC_OK;
}

extern "C" int qmc_time_stage(qmc_walkers* w, int stage, int spin, int delay_k, int reps, double* ms_per_launch) {
    if (!w || !ms_per_launch || stage < 0 || stage > 5 || spin < 0 || spin > 1 || reps < 1 || delay_k < 1 || delay_k > 128)
        return fail(QMC_ERR_ARG, "qmc_time_stage: bad argument");
    GUARD(w->sys);
    const SysDev& s = w->sys->d;
    cudaStream_t st = w->stream;
    if (s.ns[spin] == 0) return fail(QMC_ERR_ARG, "qmc_time_stage: empty spin block");
    const int kp = round_up(delay_k, 16);
    if (kp != w->d.kp) {
        int rc = alloc_window(w, kp);
        if (rc) return rc;
        CU(launch_window_reset(w->d, st));
    }
    build_lane_views(w);
    WalkDev& d = w->lane[0].d;   // what a sweep launches: the first lane's kernels (the whole crowd if it runs as one lane)
    const int p = 0, e = spin == 0 ? 0 : s.ns[0];
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    // make the inputs of the later stages valid
    CU(launch_step(s, d, spin, -1, p, 0, w->step, 0.005, 1, st));
    const int mgrid = mo_grid_for(s, spin, 5 * d.W, d.mo_grid);
    CU(launch_basis(s, d.rp, d.W, d.Phi, nullptr, st));
    CU(launch_mo(s, spin, d.Phi, 5 * d.W, d.V, d.ldv, d.mo_ws, d.mo_flags, mgrid, ++w->mo_epoch, nullptr, st));
    if (stage == 4) CU(launch_fill_int(d.mcount, d.W, delay_k, st));  // full window, S^-1 = 0: zero correction
    cudaError_t err = cudaSuccess;
    for (int r = -2; r < reps && err == cudaSuccess; r++) {
        if (r == 0) err = cudaEventRecord(e0, st);
        if (err != cudaSuccess) break;
        switch (stage) {
            case 0: err = launch_step(s, d, spin, -1, p, 0, w->step, 0.005, 1, st); break;
            case 1: err = launch_basis(s, d.rp, d.W, d.Phi, nullptr, st); break;
            case 2: err = launch_mo(s, spin, d.Phi, 5 * d.W, d.V, d.ldv, d.mo_ws, d.mo_flags, mgrid, ++w->mo_epoch, nullptr, st); break;
            case 3: err = launch_step(s, d, spin, p, p, 0, w->step, 0.005, 0, st); break;
            case 4:
                err = launch_flush(s, d, spin, st);
                if (err == cudaSuccess) err = launch_fill_int(d.mcount, d.W, delay_k, st);
                break;
            case 5: err = launch_eloc(s, d, st); break;
        }
    }
    if (err == cudaSuccess) err = cudaEventRecord(e1, st);
    if (err == cudaSuccess) err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (stage == 4) { cudaError_t e2 = launch_window_reset(w->d, st); if (err == cudaSuccess) err = e2; }
    CU(err);
    CU(cudaStreamSynchronize(st));
    *ms_per_launch = (double)ms / reps;
    return QMC_OK;
}

extern "C" int qmc_philox_words(int n, const uint32_t* ctr_key, uint32_t* out, void* cuda_stream) {
    if (n < 0 || (n > 0 && (!ctr_key || !out))) return fail(QMC_ERR_ARG, "qmc_philox_words: bad argument");
    if (n == 0) return QMC_OK;
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint32_t* buf = nullptr;
    CU(cudaMalloc((void**)&buf, (size_t)n * 10 * 4));
    cudaError_t e = cudaMemcpyAsync(buf, ctr_key, (size_t)n * 6 * 4, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = launch_philox_words(n, buf, buf + (size_t)n * 6, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out, buf + (size_t)n * 6, (size_t)n * 4 * 4, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(buf);
    CU(e);
    return QMC_OK;
}

extern "C" int qmc_measure_fp64_peak(double ms_target, double* tflops, void* cuda_stream) {
    if (!tflops || !(ms_target > 0.0)) return fail(QMC_ERR_ARG, "qmc_measure_fp64_peak: bad argument");
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = sms * 2, threads = 512, iters = 20000;
    double* buf;
    CU(cudaMalloc((void**)&buf, (size_t)grid * threads * 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaError_t err = launch_dmma_peak(buf, grid, threads, 200, st);
    const double flop_per_launch = 2.0 * 8 * 8 * 4 * 8.0 * iters * (double)grid * (threads / 32);
    double total_ms = 0.0, total_flop = 0.0;
    while (err == cudaSuccess && total_ms < ms_target) {
        err = cudaEventRecord(e0, st);
        if (err == cudaSuccess) err = launch_dmma_peak(buf, grid, threads, iters, st);
        if (err == cudaSuccess) err = cudaEventRecord(e1, st);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
        total_ms += ms;
        total_flop += flop_per_launch;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    CU(err);
    *tflops = total_flop / (total_ms * 1e-3) * 1e-12;
    return QMC_OK;
}
