#!/usr/bin/env python
"""bench.py -- electron-moves/s of the batched Slater-Jastrow move on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands, on the host cores

A "step" is ONE SWEEP of the whole hot path (rows a1-a9: drift, Philox proposal, basis, MO contraction,
ratio + Jastrow, accept/reject, delayed-update flushes, local energy) over the crowd of the 256-water
config (BASELINE.json configs[2]: 256 walkers x 2048 electrons, tau 0.005, delay_k 64) = 524,288 proposed
moves per GPU.  N > 1: one process per GPU (torchrun), each with its own 256 walkers (global walker ids
rank*256..) -- weak scaling, no data-path collective; time is the max over ranks.

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the definitions of every key.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import qmc_inputs as qi  # noqa: E402

METRIC, UNIT = "electron_moves_per_s", "moves/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--walkers", type=int, default=None, help="walkers per GPU (default: the config's)")
    ap.add_argument("--delay-k", type=int, default=None)
    ap.add_argument("--prof-stride", type=int, default=16, help="time the per-electron stages of every n-th electron")
    ap.add_argument("--config4-sweep", action="store_true",
                    help="BASELINE.json configs[4]: delay_k x crowd-size sweep on the 256-water system, 5 sweeps per point; "
                         "prints one JSON line per point and checks the accept bits against the config-2 trajectory")
    ap.add_argument("--paper-regime", action="store_true",
                    help="row f4: the paper's own regime -- water clusters of 8/16/24/152 valence electrons, 4320 walkers per GPU "
                         "(PAPER.md L279-302) -- on the one-launch small-system path and on the per-electron path; one JSON line each")
    ap.add_argument("--one-lane", action="store_true", help="QMC_ONE_LANE: the crowd as one lane (the round-1 schedule), for comparison")
    ap.add_argument("--mo-ctas", type=int, default=0, help="qmc_set_mo_ctas of the headline walker set (0 = all SMs)")
    ap.add_argument("--no-screened", action="store_true", help="skip the extra leg with QMC_SCREEN_MO")
    ap.add_argument("--no-dmc", action="store_true", help="skip the untimed row-f1 leg (one DMC generation + reconfiguration)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--crowds", action="store_true", help="also run the two-crowds leg (qmc_sweep_crowds over two walker sets; superseded by "
                                                          "the lanes inside qmc_sweep, kept for comparison)")
    ap.add_argument("--crowd-ctas", type=int, default=124, help="CTAs of each crowd's contraction in the two-crowds leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-moves", type=int, default=96, help="electron moves per walker in the CPU-baseline sample")
    return ap.parse_args()


def workload_name(wl, walkers, k):
    s = wl.system
    return (f"configs[{wl.config}] {s.name}: {s.n_elec} electrons, {s.n_basis} GTOs, {walkers} walkers/GPU, "
            f"tau {wl.tau}, delay_k {k}")


def config_dict(wl, walkers, k, world):
    """The `config` object of the JSON line -- the same keys for both arms, so that the driver's same_config check compares
    like with like (the reference arm times a bounded SAMPLE of this workload: see its cpu_baseline.sample)."""
    return dict(workload=workload_name(wl, walkers, k), step="one sweep = one proposed move per electron per walker",
                moves_per_step=walkers * wl.system.n_elec * world,
                l2="per-step working set (A^-1 + row caches, ~25 GB/GPU) >> 126 MB L2; no flush needed")


def flop_model(sysm, n_moves, n_accepted):
    """MO contraction 2*c*N_b*N_s per proposed move (c = 5) + 4*N_s^2 per accepted move."""
    ns = sysm.n_up
    return n_moves * 2.0 * 5 * sysm.n_basis * ns + n_accepted * 4.0 * ns * ns


def stage_rooflines(sysm, W, k, acc, ms, hbm_gbs, fp64_tflops):
    """Per-stage roofline fractions: ALGORITHMIC bytes or flops of ONE launch of each stage
    (what the method must move, not what the kernel happens to move) over its mean duration measured
    with CUDA events.  acc = accepted fraction; the mean number of rows pending in the delay window when a fused step
    kernel runs is mbar = acc*(k-1)/2.  The step kernel = rows a1 + a5 + a6 + a7:
        8 N_s (1 + 3 + c_r)   drift row of A^-T, three gradient rows of the row cache, c_r = 4 rows of V at r'
      + 16 mbar N_s           the window (Vbuf and Wbuf rows pending), once each
      + 24 N_e                the walker's positions (Jastrow)
      + 7 * 8 N_s acc         commit of an accepted move: five row-cache rows + two window rows written
    `impl_bytes_per_launch` is what this implementation moves by its own count (the one-pass step kernel: the algorithmic
    rows plus v_4 / a_p read a second time on accept, S^-1) -- reported beside the algorithmic figure, never used for `frac`."""
    ns, nb, ne, na = sysm.n_up, sysm.n_basis, sysm.n_elec, sysm.n_atoms
    mbar = acc * (k - 1) / 2.0
    per_walker_step = 8.0 * ns * (1 + 3 + 4) + 16.0 * mbar * ns + 24.0 * ne + 7 * 8.0 * ns * acc
    impl_step = (8.0 * ns * (4 + 1 + 1 + 3 + acc * (7 + 2))                   # V rows, a_p, a_q, gradient rows; on accept 7 rows stored, v_4 and a_p read again (L2)
                 + 16.0 * ns * mbar                                          # Wbuf and Vbuf, once each (csrc/step_onepass.cuh)
                 + 8.0 * mbar * mbar * (acc * 2 + 1)                          # S^-1 read, and rewritten on accept
                 + 24.0 * (ne + na))                                          # partner coordinates, one Jastrow pass
    m = acc * k
    alg = {
        "basis": ("hbm", 8.0 * 5 * W * nb),
        "mo": ("tensor", 2.0 * 5 * W * nb * ns),
        "step": ("hbm", W * per_walker_step),
        "flush": ("tensor", W * (4.0 * m * ns * ns + 2.0 * m * m * ns)),
        "eloc": ("hbm", W * (40.0 * ns * ne + 24.0 * ne)),
    }
    out = {}
    for st, (bound, amount) in alg.items():
        t = ms.get(st)
        if not t:
            continue
        if bound == "hbm":
            a = amount / (t * 1e-3) * 1e-9
            out[st] = dict(bound="hbm", achieved=a, peak=hbm_gbs, unit="GB/s", frac=a / hbm_gbs, bytes_per_launch=amount)
            if st == "step":
                out[st]["impl_bytes_per_launch"] = W * impl_step
        else:
            a = amount / (t * 1e-3) * 1e-12
            out[st] = dict(bound="tensor", achieved=a, peak=fp64_tflops, unit="TFLOP/s", frac=a / fp64_tflops, flop_per_launch=amount)
    return out


# ---------------------------------------------------------------------------------------- clocks

class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "200"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------- CPU oracle legs

def oracle_sample(wl, n_steps, n_warm, moves_per_step, walkers=None):
    """Time the oracle (as it stands) on the host cores: `cores` walkers in parallel, each doing
    moves_per_step electron moves of sweep 0 per step, continuing along the sweep.  Walker creation
    (all orbital rows + LU inverse) is not timed."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    cores = oracle.default_threads()
    nw = walkers or cores
    osys = oracle.OracleSystem(wl.system)
    pos = wl.positions(0, nw)
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=cores) as ex:
        ws = list(ex.map(lambda p: osys.walker(p), pos))
    t_init = time.perf_counter() - t0
    ne = wl.system.n_elec
    times = []
    e = 0
    for s in range(n_warm + n_steps):
        lo, hi = e % ne, min(e % ne + moves_per_step, ne)
        t0 = time.perf_counter()
        with ThreadPoolExecutor(max_workers=cores) as ex:
            list(ex.map(lambda a: a[1].sweep_range(wl.seed, a[0], 0, wl.tau, lo, hi), enumerate(ws)))
        dt = time.perf_counter() - t0
        if s >= n_warm:
            times.append((dt, (hi - lo) * nw))
        e += hi - lo
    tot_t = sum(t for t, _ in times)
    tot_m = sum(m for _, m in times)
    return dict(value=tot_m / tot_t, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{nw} walkers x {moves_per_step} electron moves x {n_steps} steps of sweep 0 "
                       f"(walker creation, {t_init:.1f} s, not timed)"), tot_t / max(len(times), 1)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = qi.make_workload(args.config)
    k = args.delay_k or wl.delay_k
    cb, s_per_step = oracle_sample(wl, args.steps, args.warmup, args.cpu_moves)
    line = dict(metric=METRIC, value=cb["value"], unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=s_per_step * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference",
                config=config_dict(wl, args.walkers or wl.n_walkers, k, args.gpus),
                cpu_baseline=cb,
                e2e=dict(value=cb["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------- this repo's arm

def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2504_07948_b200 import build as qbuild
    from paper_2504_07948_b200.sharding import dist_env, reduce_report, walker_slice
    rank, local_rank, world = dist_env()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", init_method="env://", device_id=torch.device("cuda", local_rank))
    if local_rank == 0:
        qbuild.build()
    if world > 1:
        dist.barrier()
    import paper_2504_07948_b200 as qb
    qb.load_library()

    wl = qi.make_workload(args.config)
    sysm = wl.system
    W = args.walkers or wl.n_walkers
    k = args.delay_k or wl.delay_k
    lo, hi = walker_slice(W, rank)
    pos_host = torch.from_numpy(qi.initial_positions(sysm, wl.config, range(lo, hi), wl.seed)).pin_memory()
    gsys = qb.qmc_init_from(sysm)
    peak = qb.qmc_measure_fp64_peak(300.0)

    # ---- device-resident run: inputs already in HBM when the timed region starts
    pos_dev = pos_host.cuda()
    base_flags = qb.QMC_ONE_LANE if args.one_lane else 0
    gw = qb.qmc_walkers_create(gsys, pos_dev, wl.seed, first_walker_id=lo, flags=base_flags)
    if args.mo_ctas:
        qb.qmc_set_mo_ctas(gw, args.mo_ctas)
    for _ in range(args.warmup):
        qb.qmc_sweep(gw, 1, wl.tau, k)
    qb.qmc_synchronize(gw)
    st0 = qb.qmc_get_stats(gw)
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = qb.qmc_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev0.record()
    qb.qmc_sweep(gw, args.steps, wl.tau, k)   # EXACTLY K steps (sweeps), enqueued on torch's current stream
    ev1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = ev0.elapsed_time(ev1)
    launches = qb.qmc_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    st1 = qb.qmc_get_stats(gw)
    eloc = qb.qmc_get_eloc(gw)[0].clone()
    dense_bits = qb.qmc_get_accept_log(gw).cpu().numpy() if not (args.no_screened and (not args.crowds)) else None
    # ---- the per-stage times come from a SECOND pass of K sweeps on the same crowd with the in-situ stage timers on (CUDA
    # events around every prof_stride-th electron's launches): the headline above is timed without that instrumentation
    qb.qmc_set_profiling(gw, args.prof_stride)
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record()
    qb.qmc_sweep(gw, args.steps, wl.tau, k)
    pe1.record()
    torch.cuda.synchronize()
    ms_profiled_pass = pe0.elapsed_time(pe1)
    stage = qb.qmc_get_stage_times(gw)
    mo_span_us, mo_span_min_us, mo_cta_us, mo_span_n = qb.qmc_get_mo_spans(gw)
    n_lanes, lane_walkers = qb.qmc_get_lanes(gw)
    qb.qmc_set_profiling(gw, 0)
    # ---- the stages one at a time: with two lanes the in-situ event times above include queueing behind the other lane's
    # kernels, so every stage's own roofline fraction is measured on a crowd of the same size moved as ONE lane (2 profiled
    # sweeps after a warm-up sweep): there the launches of a sweep are a chain and each event pair brackets one kernel alone
    if n_lanes == 2:
        gwa = qb.qmc_walkers_create(gsys, pos_dev, wl.seed, first_walker_id=lo, flags=qb.QMC_ONE_LANE)
        qb.qmc_sweep(gwa, 1, wl.tau, k)
        qb.qmc_set_profiling(gwa, args.prof_stride)
        qb.qmc_sweep(gwa, 2, wl.tau, k)
        sa = qb.qmc_get_stage_times(gwa)
        qb.qmc_walkers_destroy(gwa)
    else:
        sa = stage
    alone = {st_: (sa[st_][0] / sa[st_][1] if sa[st_][1] else None) for st_ in sa}
    n_moves = st1["proposed"] - st0["proposed"]
    n_acc = st1["accepted"] - st0["accepted"]
    assert n_moves == W * sysm.n_elec * args.steps, (n_moves, W, sysm.n_elec, args.steps)
    assert st1["nonfinite"] == 0
    red = reduce_report(ms, n_moves, float(eloc.sum()), float((eloc * eloc).sum()), W, backend_device="cuda")
    # ---- end to end through the C ABI with HOST buffers: one whole job of K sweeps (a second walker set beside the first;
    # measured straight after the device-resident run so that both see the same thermal state)
    e2e = None
    if not args.no_e2e:
        ne = sysm.n_elec
        out_pos = torch.empty((W, ne, 3), dtype=torch.float64).pin_memory()
        out_e, out_k, out_l = [torch.empty(W, dtype=torch.float64).pin_memory() for _ in range(3)]
        out_s = torch.empty(W, dtype=torch.int8).pin_memory()
        out_b = torch.empty((args.steps, ne, W), dtype=torch.uint8).pin_memory()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        gw2 = qb.qmc_walkers_create(gsys, pos_host, wl.seed, first_walker_id=lo, flags=base_flags)     # H2D of the positions inside
        qb.qmc_sweep(gw2, args.steps, wl.tau, k)
        qb.qmc_get_positions(gw2, out=out_pos)                                        # D2H, synchronous
        qb.qmc_get_eloc(gw2, out=out_e, out_kin=out_k)
        qb.qmc_get_logpsi(gw2, out=out_l, out_sign=out_s)
        qb.qmc_get_accept_log(gw2, out=out_b)
        torch.cuda.synchronize()
        t_e2e = (time.perf_counter() - t0) * 1e3
        qb.qmc_walkers_destroy(gw2)
        red2 = reduce_report(t_e2e, W * ne * args.steps, 0.0, 0.0, W, backend_device="cuda")
        d2h = out_pos.numel() * 8 + 3 * W * 8 + W + out_b.numel()
        e2e = dict(value=red2["n_moves"] / (red2["elapsed_ms"] * 1e-3), unit=UNIT,
                   h2d_bytes_per_step=pos_host.numel() * 8 // args.steps, d2h_bytes_per_step=d2h // args.steps,
                   ms_total=red2["elapsed_ms"],
                   what="qmc_walkers_create from pinned host positions (orbital rows + inverse of all Slater matrices) "
                        f"+ qmc_sweep({args.steps}) + qmc_get_{{positions,eloc,logpsi,accept_log}} into pinned host buffers")
    # ---- the same walkers as TWO crowds of W/2 on two streams, advanced together by qmc_sweep_crowds with the
    # contraction of each limited to 124 CTAs (the basis / step kernels of one crowd overlap the contraction of the
    # other).  Reported beside the headline, not as it: the headline and its roofline are the single-crowd run above.
    crowds = None
    if not (not args.crowds) and W >= 2:
        half = W // 2
        cstreams = [torch.cuda.Stream() for _ in range(2)]
        csets = []
        for c in range(2):
            a0, a1 = (0, half) if c == 0 else (half, W)
            gwc = qb.qmc_walkers_create(gsys, pos_dev[a0:a1].contiguous(), wl.seed, first_walker_id=lo + a0, stream=cstreams[c])
            qb.qmc_set_mo_ctas(gwc, args.crowd_ctas)
            csets.append(gwc)
        for _ in range(args.warmup):
            qb.qmc_sweep_crowds(csets, 1, wl.tau, k)
        torch.cuda.synchronize()
        c0 = torch.cuda.Event(enable_timing=True)
        c0.record()
        ends = []
        for st_ in cstreams:
            st_.wait_event(c0)
        qb.qmc_sweep_crowds(csets, args.steps, wl.tau, k)
        for st_ in cstreams:
            e_ = torch.cuda.Event(enable_timing=True)
            e_.record(st_)
            ends.append(e_)
        torch.cuda.synchronize()
        msc = max(c0.elapsed_time(e_) for e_ in ends)
        cb = np.concatenate([qb.qmc_get_accept_log(x).cpu().numpy() for x in csets], axis=2)
        ce = torch.cat([qb.qmc_get_eloc(x)[0] for x in csets])
        crowds = dict(value=W * sysm.n_elec * args.steps / (msc * 1e-3), unit=UNIT, ms_per_step=msc / args.steps, crowds=2,
                      walkers_per_crowd=[half, W - half], mo_ctas=args.crowd_ctas,
                      decisions_differing_from_single_crowd=(int(((cb & 1) != (dense_bits & 1)).sum()) if dense_bits is not None else None),
                      max_abs_eloc_diff_from_single_crowd=float((ce - eloc).abs().max()),
                      what="qmc_sweep_crowds over two walker sets on two streams (per GPU; rank 0's walkers); same walkers, same "
                           "random streams as the headline run; differences are stream-K rounding (row count per crowd)")
        for x in csets:
            qb.qmc_walkers_destroy(x)
    # row f1 (outside the timed region): one DMC generation + one comb reconfiguration on the same crowd
    f1 = None
    if not args.no_dmc:
        e_t = float(eloc.mean())
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        evs[0].record()
        qb.qmc_dmc_step(gw, 1, wl.tau, k, e_t, 1.0)
        evs[1].record()
        src, e_mixed = qb.qmc_branch(gw)
        evs[2].record()
        torch.cuda.synchronize()
        f1 = dict(generation_ms=evs[0].elapsed_time(evs[1]), branch_ms=evs[1].elapsed_time(evs[2]),
                  walkers_copied=int((src.cpu().numpy() != np.arange(W)).sum()), e_trial=e_t, e_mixed=e_mixed, limiter_a=1.0,
                  what="qmc_dmc_step(1) = sweep with limited drift + weight update; qmc_branch = comb + copies of A^-1 and row caches")
    # row f2, first half (outside the timed region): d ln|Psi| / d R_a of the whole crowd
    f2 = None
    if not args.no_dmc:
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        evs[0].record()
        dl = qb.qmc_get_dlogpsi_dR(gw)
        evs[1].record()
        torch.cuda.synchronize()
        msf = evs[0].elapsed_time(evs[1])
        gemm_flop = 2.0 * W * sysm.n_basis * (sysm.n_up ** 2 + sysm.n_dn ** 2)
        f2 = dict(ms=msf, gemm_tflops_lower_bound=gemm_flop / (msf * 1e-3) * 1e-12, max_abs=float(dl.abs().max()),
                  what="qmc_get_dlogpsi_dR: (C A^-1)^T as one batched DMMA GEMM per spin (2 W N_b N_s^2 flop each) + per-atom contraction; "
                       "time includes allocating and freeing the [W][N_s][N_b] scratch")
        # second half: d E_L / d R_a by eq. (4), together with the first half from the shared C A^-1
        torch.cuda.synchronize()
        evs[0].record()
        de, dl2 = qb.qmc_get_deloc_dR(gw)
        evs[1].record()
        torch.cuda.synchronize()
        msf2 = evs[0].elapsed_time(evs[1])
        flop2 = sum(2 * 2.0 * W * sysm.n_basis * n ** 2 + 2 * 2.0 * W * n ** 3 for n in (sysm.n_up, sysm.n_dn))
        f2["deloc_dR"] = dict(ms=msf2, gemm_tflops_lower_bound=flop2 / (msf2 * 1e-3) * 1e-12, max_abs=float(de.abs().max()),
                              first_half_max_abs_diff=float((dl - dl2).abs().max()),
                              what="qmc_get_deloc_dR: eq. (4); per spin C A^-1 and C X (2 W N_b N_s^2 flop each), X = A^-1 B A^-1 "
                                   "(2 x 2 W N_s^3), per-atom contraction with third derivatives of the basis functions; both halves returned")
    # row f3 (outside the timed region): non-local pseudopotential energy of the whole crowd
    f3 = None
    if not args.no_dmc:
        qb.qmc_set_ecp(gsys, qi.make_ecp(sysm))
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        evs[0].record()
        vnl, n_pairs = qb.qmc_get_vnl(gw)
        evs[1].record()
        torch.cuda.synchronize()
        ms3 = evs[0].elapsed_time(evs[1])
        npts = 12 * n_pairs
        # pairs split between the spins like the electrons; flop of the values-only contraction
        flop3 = 2.0 * npts * sysm.n_basis * (sysm.n_up + sysm.n_dn) / 2
        f3 = dict(ms=ms3, pairs=int(n_pairs), pairs_per_walker=n_pairs / W, points=int(npts), contraction_tflops_lower_bound=flop3 / (ms3 * 1e-3) * 1e-12,
                  points_per_s=npts / (ms3 * 1e-3), vnl_mean=float(vnl.mean()),
                  what="qmc_get_vnl: 12-point rotated icosahedral quadrature around every (electron, atom) pair inside the cut-offs of "
                       "qmc_inputs.make_ecp; points batched 5 W at a time through k_basis (values only) -> k_mo_streamk -> k_nl_ratio")
    qb.qmc_walkers_destroy(gw)

    # ---- the same K sweeps with the optional screening of the MO contraction (QMC_SCREEN_MO); NOT the headline value
    screened = None
    if not args.no_screened:
        gw3 = qb.qmc_walkers_create(gsys, pos_dev, wl.seed, first_walker_id=lo, flags=qb.QMC_SCREEN_MO | base_flags)
        for _ in range(args.warmup):
            qb.qmc_sweep(gw3, 1, wl.tau, k)
        w0 = qb.qmc_get_mo_work(gw3)
        ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev2.record()
        qb.qmc_sweep(gw3, args.steps, wl.tau, k)
        ev3.record()
        torch.cuda.synchronize()
        ms3 = ev2.elapsed_time(ev3)
        w1 = qb.qmc_get_mo_work(gw3)
        sb = qb.qmc_get_accept_log(gw3).cpu().numpy()
        el3 = qb.qmc_get_eloc(gw3)[0]
        screened = dict(value=W * sysm.n_elec * args.steps / (ms3 * 1e-3), unit=UNIT, ms_per_step=ms3 / args.steps,
                        theta=1e-24, stages_executed_frac=(w1[0] - w0[0]) / max(w1[1] - w0[1], 1),
                        decisions_differing_from_dense=int(((sb & 1) != (dense_bits & 1)).sum()), decisions_compared=int(sb.size),
                        max_abs_eloc_diff_from_dense=float((el3 - eloc).abs().max()),
                        what="same crowd, same sweeps, A stages of Phi whose largest |entry| is below theta not contracted "
                             "(per GPU; rank 0's crowd); the headline `value` above is the dense contraction")
        qb.qmc_walkers_destroy(gw3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    secs = red["elapsed_ms"] * 1e-3
    value = red["n_moves"] / secs
    ns, nb = sysm.n_up, sysm.n_basis
    mo_ms, mo_n = stage["mo"]
    mo_events_ms = mo_ms / max(mo_n, 1)
    # One launch contracts the rows of ONE lane.  Its duration: the kernel is persistent -- one CTA per SM it is given, equal
    # shares of the iteration space -- so a launch costs the time its CTAs are resident (mean over the CTAs of end - start,
    # %globaltimer stamps of the sampled launches of the profiled pass).  With two lanes the two contractions overlap: most
    # CTAs of a launch start when the other lane's contraction leaves its SMs, so the span of a launch (first start to last
    # end) and an event pair on its stream also count that wait; both are reported beside it.
    W_launch = sum(lane_walkers) / n_lanes
    mo_flop = 2.0 * 5 * W_launch * nb * ns
    mo_avg_ms = mo_cta_us * 1e-3 if mo_span_n else mo_events_ms
    achieved = mo_flop / (mo_avg_ms * 1e-3) * 1e-12 if mo_avg_ms else None
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "mo_kernel_traffic.json")
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(f"config{wl.config}_W{W}")
        except (OSError, ValueError):
            traffic = None
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    share = {s: stage[s][0] * (args.prof_stride if s in ("step", "basis", "mo") else 1.0) for s in stage}
    tot_share = sum(share.values()) or 1.0
    hbm_gbs = peaks.get("hbm_gbs") or 6650.0
    stage_ms = {s: (stage[s][0] / stage[s][1] if stage[s][1] else None) for s in stage}
    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
        ms_per_step=red["elapsed_ms"] / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
        dtype="f64", data="synthetic",
        config=config_dict(wl, W, k, world), prof_stride=args.prof_stride,
        clocks=clocks, e2e=e2e, gpu_launches=int(launches),
        roofline=dict(kernel="k_mo_streamk (MO contraction V = Phi*C, persistent stream-K, DMMA m8n8k4)", bound="tensor", achieved=achieved,
                      peak=peak, unit="TFLOP/s", frac=(achieved / peak) if achieved else None, traffic=traffic,
                      peak_source="FP64 DMMA issue-rate loop measured in this run (qmc_measure_fp64_peak); nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                      peak_alt_bf16_scaled=(peaks.get("bf16_tflops_sustained", 0) * 37.2 / 2250.0) or None,
                      flop_per_launch=mo_flop, ms_per_launch=mo_avg_ms, launches_timed=int(mo_span_n or mo_n),
                      ms_per_launch_stream_events=mo_events_ms,
                      ms_per_launch_span=(mo_span_us * 1e-3) if mo_span_n else None,
                      timing="mean residency of the CTAs of the sampled launches (%globaltimer stamps of every CTA; persistent kernel, equal shares); "
                             "span and stream events beside it" if mo_span_n else "CUDA events on the stream",
                      all_launches_over_elapsed=dict(
                          achieved=mo_flop * n_lanes * sysm.n_elec * args.steps / secs * 1e-12,
                          frac=mo_flop * n_lanes * sysm.n_elec * args.steps / secs * 1e-12 / peak,
                          what="flops of ALL contraction launches of the timed region over its elapsed time: the tensor-pipe rate the sweep "
                               "sustains through this kernel, every other stage and every wait included"),
                      rows_per_launch=5 * W_launch, lanes=n_lanes,
                      share_of_step=(mo_avg_ms * n_lanes * sysm.n_elec) / (red["elapsed_ms"] / args.steps)),
        fp64_tflops_model=flop_model(sysm, red["n_moves"], n_acc * world) / secs * 1e-12,
        accept_frac=n_acc / max(n_moves, 1),
        stage_ms_per_launch=stage_ms,
        stage_timing="second pass of the same K sweeps with qmc_set_profiling on (%.1f ms per sweep against %.1f unprofiled)" % (
            ms_profiled_pass / args.steps, red["elapsed_ms"] / args.steps),
        stage_roofline=stage_rooflines(sysm, W, k, n_acc / max(n_moves, 1), alone, hbm_gbs, peak),
        stage_roofline_note="every stage alone on the GPU: the same crowd moved as ONE lane (QMC_ONE_LANE, 2 profiled sweeps, in-situ CUDA events); "
                            "in the two-lane sweep the stages of the lanes overlap and their event times (stage_ms_per_launch) include queueing",
        lanes=dict(n=n_lanes, walkers=lane_walkers),
        hbm_peak_source="MEASURED_PEAKS.json hbm_gbs" if peaks.get("hbm_gbs") else "6.65 TB/s of fallback (B200_PROFILING.md)",
        stage_share={s: share[s] / tot_share for s in share},
        eloc_mean=red["e_sum"] / red["n_walkers"],
        f1_dmc=f1,
        f2_dlogpsi_dR=f2,
        f3_vnl=f3,
        two_crowds=crowds,
        screened_mo=screened,
    )
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = oracle_sample(wl, 3, 1, args.cpu_moves)[0]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_config4(args):
    """configs[4]: W in {32,128,256,512} x delay_k in {1,4,16,64,128} on the config-2 system, 5 sweeps each from the
    initial state.  Walkers w < 256 must reproduce the first 5 sweeps of the config-2 run (W = 256, k = 64) decision by
    decision (delay invariance + walker-prefix invariance, readings A13/A20); the config-2 run itself is compared with
    the oracle in tests/test_gpu_parity.py."""
    import torch
    from paper_2504_07948_b200 import build as qbuild
    torch.cuda.set_device(0)
    qbuild.build()
    import paper_2504_07948_b200 as qb
    qb.load_library()
    wl = qi.make_workload(2)
    sysm = wl.system
    T = 5
    gsys = qb.qmc_init_from(sysm)
    peak = qb.qmc_measure_fp64_peak(300.0)
    warm = qb.qmc_walkers_create(gsys, torch.from_numpy(qi.initial_positions(sysm, wl.config, range(8), wl.seed)).cuda(), wl.seed)
    for k in (1, 4, 16, 64, 128):
        qb.qmc_sweep(warm, 1, wl.tau, k)     # loads every kernel variant once
    qb.qmc_synchronize(warm)
    qb.qmc_walkers_destroy(warm)

    def run(W, k):
        pos = torch.from_numpy(qi.initial_positions(sysm, wl.config, range(W), wl.seed)).cuda()
        gw = qb.qmc_walkers_create(gsys, pos, wl.seed)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev0.record()
        qb.qmc_sweep(gw, T, wl.tau, k)
        ev1.record()
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1)
        bits = qb.qmc_get_accept_log(gw).cpu().numpy()
        st = qb.qmc_get_stats(gw)
        eloc = qb.qmc_get_eloc(gw)[0].cpu().numpy()
        qb.qmc_walkers_destroy(gw)
        return ms, bits, st, eloc

    _, ref_bits, _, ref_eloc = run(256, 64)
    for W in (32, 128, 256, 512):
        for k in (1, 4, 16, 64, 128):
            ms, bits, st, eloc = run(W, k)
            n = min(W, 256)
            a, b = bits[:, :, :n], ref_bits[:, :, :n]
            differ = (a & 1) != (b & 1)
            flagged = ((a | b) & 2) != 0
            walkers_off = int(np.any(differ, axis=(0, 1)).sum())
            moves = W * sysm.n_elec * T
            line = dict(metric=METRIC, value=moves / (ms * 1e-3), unit=UNIT, n_gpus=1, steps=T, warmup=0, ms_per_step=ms / T,
                        dtype="f64", data="synthetic",
                        config=dict(workload=f"configs[4] water256: {W} walkers, delay_k {k}, tau {wl.tau}, 5 sweeps from the initial state"),
                        fp64_tflops_model=flop_model(sysm, moves, st["accepted"]) / (ms * 1e-3) * 1e-12, fp64_peak_tflops=peak,
                        accept_frac=st["accepted"] / moves, ties=st["ties"], nonfinite=st["nonfinite"],
                        vs_config2=dict(walkers_compared=n, decisions_compared=int(a.size), decisions_differing=int(differ.sum()),
                                        first_differences_flagged_as_ties=int((differ & flagged).sum()), walkers_diverged=walkers_off,
                                        max_abs_eloc_diff=float(np.abs(eloc[:n] - ref_eloc[:n]).max())))
            print(json.dumps(line), flush=True)


def run_paper_regime(args):
    """Second workload: synthetic valence-only water clusters of the sizes of the paper's Table I
    (8, 16, 24, 152 electrons) with the paper's 4320 walkers per GPU rank and tau = 0.01.
    Systems with <= 32 electrons per spin run a whole qmc_sweep call in one launch (small_sweep.cuh); every system is
    also timed on the per-electron kernels (QMC_LARGE_PATH).  Four walkers of every run are checked against the oracle."""
    import torch
    import oracle
    from paper_2504_07948_b200 import build as qbuild
    torch.cuda.set_device(0)
    qbuild.build()
    import paper_2504_07948_b200 as qb
    qb.load_library()
    W, T, tau, seed = args.walkers or 4320, 10, 0.01, qi.MASTER_SEED
    for n_water in (1, 2, 3, 19):
        sysm = qi.water_cluster(n_water, seed, cfg=1)
        pos = qi.initial_positions(sysm, 1, range(W), seed)
        gsys = qb.qmc_init_from(sysm)
        osys = oracle.OracleSystem(sysm)
        ref = oracle.run_crowd(sysm, pos[:4], seed, range(4), 0, 2, tau, osys=osys)
        k = min(16, sysm.n_up)
        for path, flags in (("one-launch", 0), ("per-electron", qb.QMC_LARGE_PATH)):
            if path == "one-launch" and sysm.n_up > 32:
                continue
            pos_dev = torch.from_numpy(pos).cuda()
            gw = qb.qmc_walkers_create(gsys, pos_dev, seed, flags=flags)
            qb.qmc_sweep(gw, 2, tau, k)                                   # warm-up, and the parity sample
            bits = qb.qmc_get_accept_log(gw).cpu().numpy()[:, :, :4]
            differ = int(((bits & 1) != (ref["bits"] & 1)).sum())
            e_err = float(np.abs(qb.qmc_get_eloc(gw)[0].cpu().numpy()[:4] - ref["eloc"][-1]).max())
            l0 = qb.qmc_launch_count()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            ev0.record()
            qb.qmc_sweep(gw, T, tau, k)
            ev1.record()
            torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1)
            launches = qb.qmc_launch_count() - l0
            st = qb.qmc_get_stats(gw)
            qb.qmc_walkers_destroy(gw)
            moves = W * sysm.n_elec * T
            print(json.dumps(dict(metric=METRIC, value=moves / (ms * 1e-3), unit=UNIT, n_gpus=1, steps=T, warmup=2, ms_per_step=ms / T,
                                  dtype="f64", data="synthetic", path=path, gpu_launches=int(launches),
                                  walkers_per_s=W * T / (ms * 1e-3),
                                  config=dict(workload=f"{sysm.name}: {sysm.n_elec} valence electrons, {sysm.n_basis} GTOs, {W} walkers, tau {tau}, "
                                                       f"delay_k {k if path == 'per-electron' else 1}"),
                                  accept_frac=st["accepted"] / st["proposed"], nonfinite=st["nonfinite"],
                                  oracle_check=dict(walkers=4, sweeps=2, decisions_differing=differ, max_abs_eloc_diff=e_err))), flush=True)


def main():
    args = parse()
    if args.paper_regime:
        run_paper_regime(args)
    elif args.config4_sweep:
        run_config4(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
