"""bench.py -- H_eff.psi throughput of the B200 DMRG hot path (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg2] [--mode emu|fp64|tf32]

Default workload: BASELINE.json configs[2], the CAS(54,36)-shaped SU(2) system at D_SU(2) = 2048 (the
configuration the metric and the >= 50 % target are quoted on), centre bond, in the emulated-FP64 mode
(Ozaki slices on the INT8 tensor cores, kappa = 6).  A "step" is one two-site H_eff.psi
(slice psi, stage-1 and stage-2 grouped GEMMs) on seeded synthetic inputs
 with the environment operators resident in HBM.  `value` is algorithmic GFLOP/s
(FP64-equivalent): F_alg (the library's integer, pinned to the oracle's enumerator) / time.
The same line carries the native-FP64 and 3xTF32 applies of the same inputs, the Davidson time per iteration,
one renormalization, the tensor-pipe peaks measured in this run, the roofline fractions that follow from
them, the HBM-class kernels and the CPU oracle timed on the host cores.

Multi-GPU: the path does not shard in this build, so N ranks run N
independent replicas and `value` is the sum (scaling "weak").

--impl reference times the CPU oracle (oracle/, test infrastructure) as it stands on a bounded sample of the
same workload; rank 0 only; it does not load the CUDA library.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import fixtures as fx  # noqa: E402

METRIC = "heff_psi_gflops"
UNIT = "GFLOP/s"
N_PROD = {6: 21}                       # slice products of the triangular set at kappa = 6 (Appendix A6)


def make_inputs(cfg, want_V=False):
    h, V, chol = fx.make_integrals(cfg.L, cfg.n_chol, 0, cfg.hdiag, want_V=want_V)
    tabs = fx.block_tables(cfg)
    nl, nr = cfg.bond, cfg.L - cfg.bond - 2
    return dict(cfg=cfg, h=h, V=V, chol=chol, tabs=tabs, nl=nl, nr=nr)


def add_isometries(inp):
    cfg = inp["cfg"]
    inp["isoL"] = fx.random_isometries(cfg, inp["tabs"], inp["nl"], 1)
    inp["isoR"] = fx.random_isometries(cfg, inp["tabs"], inp["nr"], 1001)
    return inp


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_median": float(np.median(pw)) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- CPU oracle (cpu_baseline, --impl reference)
def _oracle_tables(inp):
    """The oracle's own block table, term list and F_alg (oracle/falg.py): no product code involved."""
    cfg, tabs, nl, nr = inp["cfg"], inp["tabs"], inp["nl"], inp["nr"]
    from oracle import falg
    if cfg.sym == 1:
        from oracle import su2, su2_loopnest as ln
        terms = ln.two_site_terms(inp["h"], inp["V"], list(range(cfg.bond)), cfg.bond, cfg.bond + 1,
                                  list(range(cfg.bond + 2, cfg.L)))
        blocks, n = su2.psi_blocks(tabs[nl], tabs[nr], cfg.N, cfg.twoS)
        tot, per, _, _ = falg.falg(terms, tabs[nl], tabs[nr], blocks, True, cfg.twoS)
    else:
        from oracle import abelian as ab, abelian_terms as at
        from oracle.fock import spin_orbital_integrals
        t, v = spin_orbital_integrals(inp["h"], inp["V"])
        so = lambda ps: [i for p in ps for i in (2 * p, 2 * p + 1)]
        terms = at.two_site_terms(t, v, so(range(cfg.bond)), cfg.bond, cfg.bond + 1, so(range(cfg.bond + 2, cfg.L)))
        blocks, n = ab.psi_block_list(tabs[nl], tabs[nr], cfg.N, cfg.twoS)
        tot, per, _, _ = falg.falg(terms, tabs[nl], tabs[nr], blocks, False)
    return blocks, n, tot, per


def _sample(blocks, n_blocks, dims, seed=3):
    sizes = blocks[:, dims[0]] * blocks[:, dims[1]]
    pick = [int(np.argmax(sizes))]
    rng = np.random.Generator(np.random.Philox(seed))
    for i in rng.permutation(len(blocks)):
        if len(pick) >= min(n_blocks, len(blocks)):
            break
        if int(i) not in pick:
            pick.append(int(i))
    return sorted(pick)


_WORK = {}


def _su2_worker(o):
    """One sampled output block of the loop-nest SU(2) oracle (oracle/su2_loopnest.py), operator blocks = seeded
    Gaussian stand-ins of the true shapes (the oracle's arithmetic does not depend on the values)."""
    from threadpoolctl import threadpool_limits
    from oracle import su2_loopnest as ln
    inp = _WORK["inp"]
    cfg, tabs, nl, nr = inp["cfg"], inp["tabs"], inp["nl"], inp["nr"]

    def standin(tab, salt):
        memo = {}

        def get(kind, k2, i, k, ib, ik):
            key = (kind, k2, i, k, ib, ik)
            if key not in memo:
                rng = np.random.Generator(np.random.Philox(key=abs(hash((salt,) + key)) % (2 ** 63)))
                memo[key] = rng.standard_normal((int(tab[ib][2]), int(tab[ik][2])))
            return memo[key]
        return get
    with threadpool_limits(limits=1):
        opsL = ln.BlockOps(tabs[nl], list(range(cfg.bond)), inp["V"], standin(tabs[nl], 0))
        opsR = ln.BlockOps(tabs[nr], list(range(cfg.bond + 2, cfg.L)), inp["V"], standin(tabs[nr], 1))
        ts = _WORK.get("ts")
        if ts is None:
            ts = ln.TwoSite(inp["h"], inp["V"], opsL, cfg.bond, cfg.bond + 1, opsR, cfg.N, cfg.twoS)
        ts.opsL, ts.opsR = opsL, opsR
        t0 = time.perf_counter()
        ts.apply_enlarged(_WORK["psi"], outputs=[o])
        return time.perf_counter() - t0


def _u1_oracle(inp):
    from oracle import abelian as ab
    cfg = inp["cfg"]
    ints = ab.Integrals(inp["h"], inp["V"])
    Lb = ab.build_block(ints, inp["tabs"], inp["isoL"], list(range(inp["nl"])), True)
    Rb = ab.build_block(ints, inp["tabs"], inp["isoR"], list(range(cfg.L - 1, cfg.bond + 1, -1)), False)
    ts = ab.TwoSite(Lb, ab.site_block(ints, cfg.bond), ab.site_block(ints, cfg.bond + 1), Rb, cfg.N, cfg.twoS)
    ts.terms()
    return ts


def _u1_worker(o):
    from threadpoolctl import threadpool_limits
    from oracle import abelian as ab
    ts = _WORK["ts"]
    iL, s1, s2, iR = (int(v) for v in ts.blocks[o][:4])
    key = (ts.A.pair_index[(iL, ab.SITE_SECTOR_OF_STATE[s1])], ts.B.pair_index[(ab.SITE_SECTOR_OF_STATE[s2], iR)])
    with threadpool_limits(limits=1):
        t0 = time.perf_counter()
        ts.apply(_WORK["psi"], only_outputs={key})
        return time.perf_counter() - t0


def time_oracle(cfg, n_blocks, passes=1):
    """The oracle as it stands on a bounded sample of output blocks of this workload, parallelised over the
    blocks with one process per host core (SURVEY.md 8(d) "CPU baseline"); flops = the oracle's own per-block
    F_alg of the sampled blocks."""
    import multiprocessing as mp
    inp = make_inputs(cfg, want_V=True)
    blocks, n, total, per = _oracle_tables(inp)
    su2 = cfg.sym == 1
    dims = (6, 7) if su2 else (4, 5)
    cores = os.cpu_count() or 1
    pick = _sample(blocks, max(n_blocks, 1), dims)
    _WORK.clear()
    _WORK.update(inp=inp, psi=fx.random_psi(n, 2))
    if su2:
        from oracle import su2_loopnest as ln
        ops0 = ln.BlockOps(inp["tabs"][inp["nl"]], list(range(cfg.bond)), inp["V"], lambda *a: None)
        ops1 = ln.BlockOps(inp["tabs"][inp["nr"]], list(range(cfg.bond + 2, cfg.L)), inp["V"], lambda *a: None)
        _WORK["ts"] = ln.TwoSite(inp["h"], inp["V"], ops0, cfg.bond, cfg.bond + 1, ops1, cfg.N, cfg.twoS)
        worker, what = _su2_worker, ("oracle/su2_loopnest.py TwoSite.apply_enlarged (c4), operator blocks = seeded Gaussian "
                                     "stand-ins of the true shapes")
    else:
        add_isometries(inp)
        _WORK["ts"] = _u1_oracle(inp)
        worker, what = _u1_worker, "oracle/abelian.py TwoSite.apply (c3) on its own renormalized environments"
    ctx = mp.get_context("fork")
    best = None
    for _ in range(max(1, passes)):
        t0 = time.perf_counter()
        with ctx.Pool(min(cores, len(pick))) as pool:
            per_block_s = pool.map(worker, pick, chunksize=1)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    f = float(per[pick].sum())
    return dict(value=f / best / 1e9, unit=UNIT, cores=min(cores, len(pick)), kind="oracle",
                sample=f"{len(pick)} of {len(blocks)} output psi blocks (seed 3, largest included) = {f / total:.4f} of F_alg "
                       f"{total}, {best:.2f} s wall with one process per block on {min(cores, len(pick))} cores (sum of block times "
                       f"{sum(per_block_s):.1f} s); {what}; numpy, 1 BLAS thread per process",
                seconds_per_pass=best, falg_oracle=int(total))


def workload_config(cfg, n_gpus, mode=None):
    symtxt = f"2Sz={cfg.twoS} U(1)xU(1) D={cfg.D}" if cfg.sym == 0 else f"2S={cfg.twoS} SU(2) D_SU(2)={cfg.D}"
    base = fx.get_config(cfg.name)
    out = {"workload": f"{cfg.name}: L={cfg.L} N={cfg.N} {symtxt} {'centre bond' if cfg.bond == base.bond else 'bond'} "
                       f"(left block {cfg.bond} orbitals), {cfg.n_chol} Cholesky vectors, seed 0/1",
           "parallelism": f"replicas x{n_gpus}", "l2": "operators + scratch exceed L2 (no flush needed)"}
    if mode:
        out["mode"] = mode
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = fx.get_config(args.config)
    if args.bond is not None:
        cfg = cfg.with_(bond=args.bond)
    cb = time_oracle(cfg, args.ref_blocks, passes=max(1, min(args.steps, 2)))
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["seconds_per_pass"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args.gpus), "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "falg_oracle": cb["falg_oracle"]}
    print(json.dumps(line))


def replica_max(x, world, device):
    """Slowest rank's time: the only exchange of the replicas-only multi-GPU mode."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(flops_per_step, ms_max, world):
    """Whole-job GFLOP/s of `world` independent replicas that each ran one step in <= ms_max."""
    return flops_per_step / (ms_max * 1e-3) / 1e9 * world


def read_traffic(cfg_name, mode):
    """DRAM bytes per launch of the dominant kernel from a committed `ncu --set full` capture of this command
    (profiles/traffic.csv: config,mode,kernel,bytes,source); None when no capture exists for this workload."""
    try:
        for ln in open(os.path.join(ROOT, "profiles", "traffic.csv")):
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 5 and f[0] == cfg_name and f[1] == mode:
                return {"kernel": f[2], "bytes": float(f[3]), "source": f[4]}
    except OSError:
        pass
    return None


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2603_28648_b200 as pkg

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = fx.get_config(args.config)
    if args.bond is not None:          # another bond of the same system (e.g. configs[4] "site 10 from the edge")
        cfg = cfg.with_(bond=args.bond)
    mode = args.mode or ("emu" if cfg.sym == 1 else "fp64")
    MODES = {"fp64": (pkg.PREC_FP64, 0), "emu": (pkg.PREC_FP64_EMU, 6), "tf32": (pkg.PREC_TF32X3, 0),
             "perf": (pkg.PREC_FP64_EMU_PERF, 6)}      # perf: the paper's performant mode (slice products per task class)
    inp = add_isometries(make_inputs(cfg))
    stream = torch.cuda.current_stream()
    d = pkg.Dmrg(local, stream.cuda_stream)
    d.init_integrals(inp["h"], None, inp["chol"], 0.0, cfg.N, cfg.twoS, cfg.sym, cfg.D)
    d.set_mps(cfg.bond, inp["tabs"][:inp["nl"] + 1], [x[1] for x in inp["isoL"]],
              inp["tabs"][:inp["nr"] + 1], [x[1] for x in inp["isoR"]])
    t0 = time.perf_counter()
    d.build_env()
    torch.cuda.synchronize()
    build_env_s = time.perf_counter() - t0
    n = d.psi_length()
    falg = int(d.table(pkg.TAB_FALG)[0])
    psi = torch.from_numpy(fx.random_psi(n, 2)).cuda()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    # tensor-pipe peaks of this GPU with the library's full-tile micro-kernels, before the timed region
    # (clocks sampled around them: the DMMA rate depends on the power state the chip is in)
    def peaks():
        s = ClockSampler(local).start()
        out = {"fp64_dmma_tflops": d.measure_peak(pkg.PREC_FP64) / 1e12, "int8_pops": d.measure_peak(pkg.PREC_FP64_EMU) / 1e15,
               "tf32_tflops": d.measure_peak(pkg.PREC_TF32X3) / 1e12, "fp64_vector_fma_tflops": d.measure_peak(3) / 1e12}
        out["clocks"] = s.stop()
        return out
    peaks_before = peaks()

    def timed_apply(m, K, W, sample_clocks=False):
        prec, kap = MODES[m]
        out = torch.empty_like(psi)
        for _ in range(W):
            d.heff_apply(psi, out, prec, kap)                  # the first call re-plans and slices the operators
        sampler = ClockSampler(local) if sample_clocks else None
        barrier()
        if sampler:
            sampler.start()
        barrier()
        lc0 = d.launch_count()
        e0.record(stream)
        for _ in range(K):
            d.heff_apply(psi, out, prec, kap)
        e1.record(stream)
        launches = d.launch_count() - lc0                      # counted by the library at its launch sites
        barrier()
        ms = replica_max(e0.elapsed_time(e1), world, "cuda") / K
        clocks = sampler.stop() if sampler else None
        counts = d.table(pkg.TAB_COUNTS)
        d.set_timing(True)
        s1, s2, sl, i8, t1 = [], [], [], [], []
        for _ in range(3):
            d.heff_apply(psi, out, prec, kap)
            a, b = d.last_stage_ms()
            s1.append(a); s2.append(b)
            if m != "fp64":
                a, b = d.last_emu_ms()
                sl.append(a); i8.append(b); t1.append(d.last_emu_stage1_ms())
        d.set_timing(False)
        r = {"ms_per_apply": ms, "gflops": falg / (ms * 1e-3) / 1e9, "stage1_ms": float(np.mean(s1)), "stage2_ms": float(np.mean(s2)),
             "stage1_flops": int(counts[11]), "stage2_flops": int(counts[12]), "passes": int(counts[14]),
             "launches_per_apply": launches / K, "launches_timed": int(launches)}
        if m != "fp64":
            r.update(stage2_slice_T_ms=float(np.mean(sl)), stage2_tensor_kernel_ms=float(np.mean(i8)),
                     stage1_tensor_kernel_ms=float(np.mean(t1)),
                     tensor_flops_stage1=int(counts[18]), tensor_flops_stage2=int(counts[15]),
                     tensor_share_of_falg=(int(counts[18]) + int(counts[15])) / falg)
            if m == "perf":
                kept, eager = d.last_emu_products()
                r["stage2_slice_products_kept_over_eager"] = kept / eager if eager else None
        return r, out, clocks

    K, W = args.steps, max(args.warmup, 3)
    results = {}
    order = [m for m in ("fp64", "tf32", "perf", "emu") if m != mode] + [mode]      # the headline mode last: its plan stays
    ref_out = None
    for m in order:
        try:
            if m == mode:
                results[m], out_m, clocks = timed_apply(m, K, W, sample_clocks=True)
            else:
                results[m], out_m, _ = timed_apply(m, max(3, min(K, 5)), 3)
            if m == "fp64":
                ref_out = out_m.clone()
            elif ref_out is not None:
                results[m]["rel_err_vs_native"] = float(torch.linalg.norm(out_m - ref_out) / torch.linalg.norm(ref_out))
            del out_m
        except pkg.DmrgError as exc:
            results[m] = {"unavailable": str(exc)}
            if m == mode:
                raise
    head = results[mode]
    ms = head["ms_per_apply"]
    prec, kap = MODES[mode]

    # end to end through host buffers (pinned), copies inside the timed region, headline mode
    hin = torch.from_numpy(fx.random_psi(n, 2)).pin_memory()
    hout = torch.empty(n, dtype=torch.float64).pin_memory()
    for _ in range(3):
        d.heff_apply_host(hin, hout, prec, kap)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        d.heff_apply_host(hin, hout, prec, kap)
    torch.cuda.synchronize()
    e2e_ms = replica_max((time.perf_counter() - t0) * 1e3, world, "cuda") / K

    # Davidson step (a7 + a8 around a4-a6), headline mode, BASELINE.json configs[2]: 10 iterations
    nit = 10 if cfg.sym == 1 else 8
    x = psi.clone()
    d.davidson_step(x, 2, 0.0, prec, kap)
    x.copy_(psi)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    theta, resid = d.davidson_step(x, nit, 0.0, prec, kap)
    dav_s = (time.perf_counter() - t0) / nit
    del x
    peaks_after = peaks()

    mp_peaks = {}
    try:
        mp_peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm_peak = mp_peaks.get("hbm_gbs") or 6500.0       # measured copy bandwidth of this pool's B200s; fallback: B200_PROFILING.md
    # HBM-class kernels (rows a4, a7, a8), each timed alone: achieved GB/s = algorithmic bytes / CUDA-event time
    try:
        hbm = d.measure_hbm_kernels(psi, nit)
        for v in hbm.values():
            v["frac_of_hbm_peak"] = v["GBps"] / hbm_peak
        hbm["peak_GBps"] = hbm_peak
        hbm["peak_source"] = "MEASURED_PEAKS.json hbm_gbs" if mp_peaks.get("hbm_gbs") else "fallback 6500 GB/s (B200_PROFILING.md)"
    except pkg.DmrgError as exc:
        hbm = {"unavailable": str(exc)}

    # one renormalization of the enlarged block (a3 + a9) in every precision mode; a fresh environment per mode
    rng = np.random.Generator(np.random.Philox(77))
    tabs = inp["tabs"]
    _, iso_next = fx.random_isometry(cfg.sym, tabs[inp["nl"]], tabs[inp["nl"] + 1], rng)
    iso_dev = torch.from_numpy(iso_next).cuda()
    renorm = {}
    for mi, m in enumerate(("fp64", "emu", "tf32")):
        try:
            if mi > 0:
                d.build_env()
            pr, kp = MODES[m]
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            d.renormalize(pkg.LEFT_TO_RIGHT, tabs[inp["nl"] + 1], iso_dev, on_device=True, precision=pr, slices=kp)
            torch.cuda.synchronize()
            renorm[m] = time.perf_counter() - t0
        except pkg.DmrgError as exc:
            renorm[m] = str(exc)
    renorm_s = renorm.get(mode)
    d.close()

    # peaks used as denominators: the larger of the two in-run readings (a kernel timed alone: burst figure)
    pk = {k: max(peaks_before[k], peaks_after[k]) for k in ("fp64_dmma_tflops", "int8_pops", "tf32_tflops")}
    # dominant kernel of the headline mode and its tensor-pipe fraction
    if mode in ("emu", "perf"):
        nprod = N_PROD[6]
        k1_ms = head["stage1_tensor_kernel_ms"]
        k2_ms = head["stage2_tensor_kernel_ms"]
        dom = "stage2" if k2_ms >= k1_ms else "stage1"
        dflops = head["tensor_flops_stage2"] if dom == "stage2" else head["tensor_flops_stage1"]
        dms = k2_ms if dom == "stage2" else k1_ms
        achieved = nprod * dflops / (dms * 1e-3) / 1e12
        peak = pk["int8_pops"] * 1e3
        kname = "k_emu_s1<6>" if dom == "stage1" else "k_emu_seg<6>"
        roofline = {"bound": "tensor", "kernel": f"{kname} ({dom} launches of the apply; tcgen05 kind::i8, {nprod} slice products per k)",
                    "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "unit_note": "INT8 tera-operations per second",
                    "frac": achieved / peak, "peak_source": "dmrg_measure_peak(INT8) in this run (library's full-tile tcgen05 kind::i8 kernel)",
                    "whole_apply_frac": nprod * falg / (ms * 1e-3) / (pk["int8_pops"] * 1e15),
                    "whole_apply_note": "north-star figure: 21 F_alg / t / P_INT8 over the whole apply (slicing, FP64 remainder and reduction included)"}
    elif mode == "tf32":
        dms, dflops = head["stage2_tensor_kernel_ms"], head["tensor_flops_stage2"]
        achieved = 3 * dflops / (dms * 1e-3) / 1e12
        roofline = {"bound": "tensor", "kernel": "k_tf32_seg (stage-2 launch; tcgen05 kind::tf32, 3 products)", "achieved": achieved,
                    "peak": pk["tf32_tflops"], "unit": "TFLOP/s", "frac": achieved / pk["tf32_tflops"],
                    "peak_source": "dmrg_measure_peak(TF32) in this run",
                    "whole_apply_frac": 3 * falg / (ms * 1e-3) / (pk["tf32_tflops"] * 1e12)}
    else:
        dom = "stage2" if head["stage2_ms"] >= head["stage1_ms"] else "stage1"
        dms, dflops = head[dom + "_ms"], head[dom + "_flops"]
        achieved = dflops / (dms * 1e-3) / 1e12
        roofline = {"bound": "tensor", "kernel": f"k_gemm_f64 ({dom} launch; DMMA.8x8x4)", "achieved": achieved,
                    "peak": pk["fp64_dmma_tflops"], "unit": "TFLOP/s", "frac": achieved / pk["fp64_dmma_tflops"],
                    "peak_source": "dmrg_measure_peak(FP64) in this run (register-resident DMMA loop)",
                    "whole_apply_frac": falg / (ms * 1e-3) / (pk["fp64_dmma_tflops"] * 1e12)}
    tr = read_traffic(cfg.name, mode) if args.bond is None else None
    roofline["traffic"] = tr["bytes"] if tr else None
    if tr:
        roofline["traffic_source"] = f"{tr['source']} ({tr['kernel']})"
    roofline["side_note_bf16_ratio_peak_tflops"] = (mp_peaks.get("bf16_tflops_sustained") or 1400.0) * 40.0 / 2250.0

    # fractions of every mode against its own in-run peak (SURVEY.md 8(d) "Reported per config and mode")
    if "ms_per_apply" in results.get("fp64", {}):
        results["fp64"]["frac_of_dmma_peak_whole_apply"] = results["fp64"]["gflops"] / 1e3 / pk["fp64_dmma_tflops"]
    if "ms_per_apply" in results.get("emu", {}):
        results["emu"]["int8_pipe_frac_whole_apply"] = 21 * results["emu"]["gflops"] * 1e9 / (pk["int8_pops"] * 1e15)
        results["emu"]["kappa"] = 6
    if "ms_per_apply" in results.get("tf32", {}):
        results["tf32"]["tf32_pipe_frac_whole_apply"] = 3 * results["tf32"]["gflops"] * 1e9 / (pk["tf32_tflops"] * 1e12)
    if "ms_per_apply" in results.get("fp64", {}):
        for m in ("emu", "perf", "tf32"):
            if "ms_per_apply" in results.get(m, {}):
                results[m]["speedup_vs_native"] = results["fp64"]["ms_per_apply"] / results[m]["ms_per_apply"]

    if "ms_per_apply" in results.get("perf", {}):
        # against the eager product count 21 F_alg, as for "emu": the mode does the same job with fewer products
        results["perf"]["int8_pipe_frac_whole_apply_at_eager_count"] = 21 * results["perf"]["gflops"] * 1e9 / (pk["int8_pops"] * 1e15)
        results["perf"]["kappa"] = 6
    dtype = {"emu": "f64 emulated on int8 slices (Ozaki, kappa=6, int32 accumulation, f64 recombination)", "fp64": "f64",
             "perf": "f64 emulated on int8 slices (Ozaki, kappa=6 storage, slice products per task class from the exponent spread)",
             "tf32": "tf32x3 (f32 accumulation)"}[mode]
    line = {"metric": METRIC, "value": replica_throughput(falg, ms, world), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": dtype,
            "data": "synthetic", "config": workload_config(cfg, world, mode), "clocks": clocks,
            "e2e": {"value": falg / (e2e_ms * 1e-3) / 1e9 * world, "unit": UNIT, "h2d_bytes_per_step": 8 * n,
                    "d2h_bytes_per_step": 8 * n, "ms_per_step": e2e_ms},
            "gpu_launches": head["launches_timed"], "roofline": roofline, "falg_per_apply": falg, "psi_len": n,
            "modes": results, "peaks_measured": {"before": peaks_before, "after": peaks_after, "used": pk},
            "davidson": {"s_per_iter": dav_s, "n_iter": nit, "mode": mode, "theta_last": float(theta[-1]), "resid_last": float(resid[-1])},
            "renormalize_s": renorm_s, "renormalize_s_by_mode": renorm, "build_env_s": build_env_s, "hbm_kernels": hbm}
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            cb = time_oracle(cfg, args.ref_blocks)
            line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
            line["falg_oracle"] = cb["falg_oracle"]
            line["falg_matches_oracle"] = cb["falg_oracle"] == falg
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg2")
    ap.add_argument("--mode", default=None, choices=["emu", "fp64", "tf32", "perf"],
                    help="headline precision mode (default: emu for the SU(2) configs, fp64 for the abelian ones)")
    ap.add_argument("--bond", type=int, default=None, help="left-block size, overrides the config's centre bond")
    ap.add_argument("--ref-blocks", type=int, default=16, help="output blocks in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
