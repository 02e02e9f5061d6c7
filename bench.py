"""bench.py -- H_eff.psi throughput of the B200 DMRG hot path (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg1]

A "step" is one two-site H_eff.psi application (SURVEY.md 8(a) rows a5 + a6: stage-1 and
stage-2 grouped GEMMs) at the centre bond of the configuration, on seeded synthetic inputs
 with the environment operators resident in HBM.  `value` is
algorithmic GFLOP/s: F_alg (reported by the library as an integer) / time.
The JSON line also carries the Davidson time per iteration (rows a7, a8), one renormalization
(rows a3, a9), the roofline of the dominant kernel and the CPU oracle timed on the host cores.

Multi-GPU: the path does not shard in this build, so
N ranks run N independent replicas and `value` is the sum (scaling "weak").

--impl reference times the CPU oracle (oracle/, test infrastructure) as it stands on a bounded
sample of the same workload; rank 0 only.
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
# nominal dense tensor peaks per GPU used only for the dtype ratio (B200_PROFILING.md table; FP64
# tensor 40 TFLOP/s is the HGX B200 data-sheet figure quoted in SURVEY.md section 7)
NOMINAL_BF16_TF, NOMINAL_FP64_TF = 2250.0, 40.0


def make_inputs(cfg):
    h, _, chol = fx.make_integrals(cfg.L, cfg.n_chol, 0, cfg.hdiag, want_V=False)
    tabs = fx.block_tables(cfg)
    nl, nr = cfg.bond, cfg.L - cfg.bond - 2
    isoL = fx.random_isometries(cfg, tabs, nl, 1)
    isoR = fx.random_isometries(cfg, tabs, nr, 1001)
    return dict(cfg=cfg, h=h, chol=chol, tabs=tabs, nl=nl, nr=nr, isoL=isoL, isoR=isoR)


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

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(inp, n_sample_blocks, seed=3):
    """Oracle environment + a seeded sample of output blocks (largest always included)."""
    from oracle import abelian as ab
    cfg = inp["cfg"]
    V = np.einsum("cij,ckl->ijkl", inp["chol"], inp["chol"])
    ints = ab.Integrals(inp["h"], V)
    Lb = ab.build_block(ints, inp["tabs"], inp["isoL"], list(range(inp["nl"])), True)
    Rb = ab.build_block(ints, inp["tabs"], inp["isoR"], list(range(cfg.L - 1, cfg.bond + 1, -1)), False)
    ts = ab.TwoSite(Lb, ab.site_block(ints, cfg.bond), ab.site_block(ints, cfg.bond + 1), Rb, cfg.N, cfg.twoS)
    ts.terms()
    nb = len(ts.blocks)
    rng = np.random.Generator(np.random.Philox(seed))
    sizes = ts.blocks[:, 4] * ts.blocks[:, 5]
    pick = {int(np.argmax(sizes))}
    for i in rng.permutation(nb):
        if len(pick) >= min(n_sample_blocks, nb):
            break
        pick.add(int(i))
    pick = sorted(pick)
    keys = set()
    for i in pick:
        iL, s1, s2, iR = (int(v) for v in ts.blocks[i][:4])
        keys.add((ts.A.pair_index[(iL, ab.SITE_SECTOR_OF_STATE[s1])], ts.B.pair_index[(ab.SITE_SECTOR_OF_STATE[s2], iR)]))
    return ts, pick, keys


def falg_tables(inp):
    """F_alg per output block from a planning context (integer tables only, no GPU work)."""
    import paper_2603_28648_b200 as pkg
    cfg = inp["cfg"]
    d = pkg.Dmrg(-1)
    d.init_integrals(inp["h"], None, inp["chol"], 0.0, cfg.N, cfg.twoS, cfg.sym, cfg.D)
    d.set_mps(cfg.bond, inp["tabs"][:inp["nl"] + 1], [], inp["tabs"][:inp["nr"] + 1], [])
    d.plan_bond()
    per_block = d.table(pkg.TAB_FALG_BLOCKS)
    total = int(d.table(pkg.TAB_FALG)[0])
    d.close()
    return per_block, total


def time_oracle_su2(inp, steps, warmup):
    """SU(2) configs: the expansion oracle (oracle/su2.py) cannot reach the full size, so the bounded
    sample is the same recipe scaled down (L=12, same filling and spin, D_SU(2)=48)."""
    from threadpoolctl import threadpool_limits
    from oracle import su2
    big = inp["cfg"]
    Ls = 12
    Ns = 2 * ((big.N * Ls) // (2 * big.L)) + (big.twoS % 2)
    cfg = big.with_(name=big.name + "_sample", L=Ls, N=Ns, D=48, bond=Ls // 2 - 1, n_chol=8, twoS=big.twoS % 2 + (2 if big.twoS >= 2 else 0))
    small = make_inputs(cfg)
    _, total = falg_tables(small)
    V = np.einsum("cij,ckl->ijkl", small["chol"], small["chol"])
    with threadpool_limits(limits=1):
        ex = su2.ExpandedTwoSite(small["h"], V, cfg.N, cfg.twoS, cfg.bond, small["tabs"][:small["nl"] + 1],
                                 small["isoL"], small["tabs"][:small["nr"] + 1], small["isoR"])
        psi = fx.random_psi(ex.n, 2)
        ex.apply(psi)
        for _ in range(warmup):
            ex.apply(psi)
        t0 = time.perf_counter()
        for _ in range(steps):
            ex.apply(psi)
        dt = (time.perf_counter() - t0) / steps
    return dict(value=total / dt / 1e9, unit=UNIT, cores=1, kind="oracle",
                sample=f"scaled-down {cfg.name}: L={cfg.L} N={cfg.N} 2S={cfg.twoS} D_SU(2)={cfg.D} (F_alg {total:.3g}), "
                       f"{dt:.2f} s per pass; oracle/su2.py expansion into oracle/abelian.py, numpy, 1 thread",
                seconds_per_pass=dt)


def time_oracle(inp, steps, warmup, n_sample_blocks):
    if inp["cfg"].sym == 1:
        return time_oracle_su2(inp, steps, warmup)
    from threadpoolctl import threadpool_limits
    per_block, total = falg_tables(inp)
    with threadpool_limits(limits=1):
        ts, pick, keys = oracle_sample(inp, n_sample_blocks)
        psi = fx.random_psi(ts.n, 2)
        for _ in range(warmup):
            ts.apply(psi, only_outputs=keys)
        t0 = time.perf_counter()
        for _ in range(steps):
            ts.apply(psi, only_outputs=keys)
        dt = (time.perf_counter() - t0) / steps
    f = float(per_block[pick].sum())
    return dict(value=f / dt / 1e9, unit=UNIT, cores=1, kind="oracle",
                sample=f"{len(pick)} of {len(ts.blocks)} output psi blocks (seed 3, largest included) = "
                       f"{f / total:.3f} of F_alg, {dt:.2f} s per pass; oracle/abelian.py TwoSite.apply, numpy, 1 thread",
                seconds_per_pass=dt)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = fx.get_config(args.config)
    if args.bond is not None:
        cfg = cfg.with_(bond=args.bond)
    inp = make_inputs(cfg)
    cb = time_oracle(inp, args.steps, args.warmup, args.ref_blocks)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["seconds_per_pass"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args.gpus), "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def workload_config(cfg, n_gpus):
    symtxt = f"2Sz={cfg.twoS} U(1)xU(1) D={cfg.D}" if cfg.sym == 0 else f"2S={cfg.twoS} SU(2) D_SU(2)={cfg.D}"
    return {"workload": f"{cfg.name}: L={cfg.L} N={cfg.N} {symtxt} {'centre bond' if cfg.bond == fx.get_config(cfg.name).bond else 'bond'} "
                        f"(left block {cfg.bond} orbitals), {cfg.n_chol} Cholesky vectors, seed 0/1",
            "parallelism": f"replicas x{n_gpus}", "l2": "operators + scratch exceed L2 (no flush needed)"}


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

    def max_over_ranks(x):
        return replica_max(x, world, "cuda")

    cfg = fx.get_config(args.config)
    if args.bond is not None:          # measure another bond of the same system (e.g. configs[4] "site 10 from the edge")
        cfg = cfg.with_(bond=args.bond)
    inp = make_inputs(cfg)
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
    counts = d.table(pkg.TAB_COUNTS)
    psi = torch.from_numpy(fx.random_psi(n, 2)).cuda()
    out = torch.empty_like(psi)

    K, W = args.steps, max(args.warmup, 3)
    for _ in range(W):
        d.heff_apply(psi, out)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(K):
        d.heff_apply(psi, out)
    e1.record(stream)
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1)) / K
    clocks = sampler.stop()

    # per-kernel durations of the same launches, CUDA events on the library's stream
    d.set_timing(True)
    s1, s2 = [], []
    for _ in range(max(3, min(K, 10))):
        d.heff_apply(psi, out)
        a, b = d.last_stage_ms()
        s1.append(a); s2.append(b)
    d.set_timing(False)
    ms1, ms2 = float(np.mean(s1)), float(np.mean(s2))

    # end to end through host buffers (pinned), copies inside the timed region
    hin = torch.from_numpy(fx.random_psi(n, 2)).pin_memory()
    hout = torch.empty(n, dtype=torch.float64).pin_memory()
    for _ in range(3):
        d.heff_apply_host(hin, hout)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        d.heff_apply_host(hin, hout)
    torch.cuda.synchronize()
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3) / K

    # Davidson step (a7 + a8 around a5/a6) and one renormalization (a3 + a9)
    nit = 8
    x = psi.clone()
    d.davidson_step(x, nit)
    x.copy_(psi)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    theta, resid = d.davidson_step(x, nit)
    dav_s = (time.perf_counter() - t0) / nit
    peak_fp64 = d.measure_peak(pkg.PREC_FP64)
    # emulated-FP64 engine (Ozaki over INT8 tcgen05): tensor-pipe peak and the standalone GEMM on a
    # shape of this workload's size class
    peak_i8 = d.measure_peak(pkg.PREC_FP64_EMU)
    peak_dfma = d.measure_peak(3)     # FP64 vector FMA rate (the emulated epilogue's unit)
    eM, eN, eK = 4096, 4096, 4096
    eA = torch.randn(eM, eK, dtype=torch.float64, device="cuda")
    eB = torch.randn(eK, eN, dtype=torch.float64, device="cuda")
    eC = torch.empty(eM, eN, dtype=torch.float64, device="cuda")
    d.emu_gemm(eM, eN, eK, eA, eB, eC, 6)
    e_slice_ms, e_gemm_ms = d.emu_gemm(eM, eN, eK, eA, eB, eC, 6)
    e_ref = eA @ eB
    e_err = float(torch.linalg.norm(eC - e_ref) / torch.linalg.norm(e_ref))
    emu = {"engine": "dmrg_emu_gemm (k_emu_seg<6>: 21 slice products as 8 stacked-N tcgen05 kind::i8 MMAs per k step, bulk-copy pipeline)", "shape": [eM, eN, eK],
           "gemm_ms": e_gemm_ms, "slice_ms": e_slice_ms, "fp64_equiv_tflops": 2.0 * eM * eN * eK / e_gemm_ms / 1e9,
           "int8_pops": 21 * 2.0 * eM * eN * eK / (e_gemm_ms * 1e-3) / 1e15, "int8_peak_pops_measured": peak_i8 / 1e15,
           "tensor_pipe_frac": 21 * 2.0 * eM * eN * eK / (e_gemm_ms * 1e-3) / peak_i8, "rel_err_vs_fp64": e_err,
           "fp64_vector_fma_tflops_measured": peak_dfma / 1e12}
    del eA, eB, eC, e_ref
    # H_eff.psi of the same workload in emulated mode (kappa = 6: stage-1 jobs and stage-2 segments of the large
    # sector pairs on the INT8 tensor cores, the small ones stay native FP64), SURVEY.md 8(d) "Reported per config and mode"
    def reduced_mode(prec, kap, n_prod, peak_ops):
        """One reduced-precision mode on the same inputs: ms per apply, stage split, error against native."""
        try:
            out_e = torch.empty_like(psi)
            for _ in range(3):
                d.heff_apply(psi, out_e, prec, kap)       # the first call re-plans and slices the operators
            ce = d.table(pkg.TAB_COUNTS)
            reps = max(3, min(K, 10))
            e0.record(stream)
            for _ in range(reps):
                d.heff_apply(psi, out_e, prec, kap)
            e1.record(stream)
            torch.cuda.synchronize()
            emu_ms = e0.elapsed_time(e1) / reps
            d.set_timing(True)
            d.heff_apply(psi, out_e, prec, kap)
            (em1, em2), (esl, ei8) = d.last_stage_ms(), d.last_emu_ms()
            d.set_timing(False)
            f2, f1 = float(ce[15]), float(ce[18])
            r = {"ms_per_apply": emu_ms, "gflops_fp64_equiv": falg / (emu_ms * 1e-3) / 1e9,
                 "speedup_vs_native": ms / emu_ms,
                 "rel_err_vs_native": float(torch.linalg.norm(out_e - out) / torch.linalg.norm(out)),
                 "stage1_ms": em1, "stage2_ms": em2, "stage2_slice_T_ms": esl, "stage2_tensor_kernel_ms": ei8,
                 "tensor_flops_stage1": f1, "tensor_flops_stage2": f2, "tensor_share_of_falg": (f1 + f2) / falg,
                 "stage2_tensor_kernel_fp64_equiv_tflops": f2 / (ei8 * 1e-3) / 1e12 if ei8 > 0 else None,
                 # whole apply against the tensor pipe of the mode: n_prod * F_alg / t / peak
                 "tensor_pipe_frac_whole_apply": n_prod * falg / (emu_ms * 1e-3) / peak_ops if peak_ops else None,
                 "segments": int(ce[16]), "tiles": int(ce[17]), "passes": int(ce[14])}
            xe = psi.clone()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            th_e, rs_e = d.davidson_step(xe, nit, 0.0, prec, kap)
            r["davidson_s_per_iter"] = (time.perf_counter() - t0) / nit
            # The first Ritz value is <psi|H|psi>; later ones differ more because the preconditioner r_i / (theta - diag_i)
            # amplifies rounding differences 10-500x per iteration on random environments
            r["davidson_theta_minus_native_iter1"] = float(th_e[0] - theta[0])
            r["davidson_theta_minus_native_last"] = float(th_e[-1] - theta[-1])
            del out_e, xe
            return r
        except pkg.DmrgError as exc:
            return {"unavailable": str(exc)}

    emu_heff = reduced_mode(pkg.PREC_FP64_EMU, 6, 21, peak_i8)
    emu_heff["kappa"] = 6
    # 3xTF32 (hi/lo split, three tcgen05 kind::tf32 products, FP32 accumulation; tolerance 1e-5); the fraction is
    # against the TF32 rate of the library's full-tile micro-kernel measured in this run
    peak_tf32 = d.measure_peak(pkg.PREC_TF32X3)
    tf32_heff = reduced_mode(pkg.PREC_TF32X3, 0, 3, peak_tf32)
    tf32_heff["tf32_peak_measured_tflops"] = peak_tf32 / 1e12
    try:
        d.heff_apply(psi, out)                                      # back to the native plan
    except pkg.DmrgError:                                           # a reduced mode that ran out of memory leaves no plan
        d.build_env()
        d.heff_apply(psi, out)
    emu["heff_apply"] = emu_heff
    rng = np.random.Generator(np.random.Philox(77))
    tabs = inp["tabs"]
    _, iso_next = fx.random_isometry(cfg.sym, tabs[inp["nl"]], tabs[inp["nl"] + 1], rng)
    iso_dev = torch.from_numpy(iso_next).cuda()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    d.renormalize(pkg.LEFT_TO_RIGHT, tabs[inp["nl"] + 1], iso_dev, on_device=True)
    torch.cuda.synchronize()
    renorm_s = time.perf_counter() - t0
    d.close()

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    bf16 = peaks.get("bf16_tflops_sustained") or peaks.get("bf16_tflops")
    src = "measured bf16 (MEASURED_PEAKS.json, sustained) x nominal FP64/bf16 ratio 40/2250"
    if not bf16:
        bf16, src = 1400.0, "fallback bf16 1.4 PFLOP/s sustained (B200_PROFILING.md) x nominal ratio 40/2250"
    peak_tf = bf16 * NOMINAL_FP64_TF / NOMINAL_BF16_TF
    # dominant kernel: the stage-2 launch of k_gemm_f64 (half of F_alg, the longer of the two)
    f1, f2 = float(counts[11]), float(counts[12])          # algorithmic flops of the two launches
    dom_ms, dom, dom_f = (ms2, "stage2", f2) if ms2 >= ms1 else (ms1, "stage1", f1)
    achieved_tf = dom_f / (dom_ms * 1e-3) / 1e12
    # DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` captures of the same command
    # (profiles/r1_ncu_stage_kernels.txt: dram__bytes_read.sum + dram__bytes_write.sum); null where no capture exists
    ncu_traffic = {("cfg1", "stage1"): 434.701568e6 + 1.930675e9, ("cfg1", "stage2"): 2.614642e9 + 18.599168e6,
                   ("cfg1_d2048", "stage2"): 117.734419e9 + 69.211136e6}
    roofline = {"bound": "tensor", "kernel": f"k_gemm_f64<2> ({dom} launch)", "achieved": achieved_tf, "peak": peak_tf,
                "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
                "traffic": ncu_traffic.get((cfg.name, dom)) if args.bond is None else None, "peak_source": src,
                "fp64_dmma_microbench_tflops": peak_fp64 / 1e12,
                "frac_of_microbench": achieved_tf / (peak_fp64 / 1e12),
                "stage1_ms": ms1, "stage2_ms": ms2, "stage1_flops": f1, "stage2_flops": f2}

    gflops = replica_throughput(falg, ms, world)
    line = {"metric": METRIC, "value": gflops, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(cfg, world), "clocks": clocks,
            "e2e": {"value": falg / (e2e_ms * 1e-3) / 1e9 * world, "unit": UNIT, "h2d_bytes_per_step": 8 * n,
                    "d2h_bytes_per_step": 8 * n, "ms_per_step": e2e_ms},
            # per apply: one stage-1 and one stage-2 launch per pass, plus the split-K reduction when any block is chunked
            "gpu_launches": K * (2 * int(counts[14]) + (1 if counts[13] > 0 else 0)), "roofline": roofline,
            "falg_per_apply": falg, "psi_len": n,
            "davidson": {"s_per_iter": dav_s, "n_iter": nit, "theta_last": float(theta[-1]), "resid_last": float(resid[-1])},
            "renormalize_s": renorm_s, "build_env_s": build_env_s, "emulated_fp64_engine": emu, "tf32x3": {"heff_apply": tf32_heff},
            "plan": {"stage1_jobs": int(counts[0]), "stage2_segments": int(counts[3]), "stage1_tiles": int(counts[4]),
                     "stage2_tiles": int(counts[5]), "scratch_GB": float(counts[6]) * 8 / 1e9,
                     "operator_GB": float(counts[7] + counts[8] + counts[9] + counts[10]) * 8 / 1e9}}
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            cb = time_oracle(inp, 1, 0, 10 ** 9)       # one full pass over every output block
            line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg1")
    ap.add_argument("--bond", type=int, default=None, help="left-block size, overrides the config's centre bond")
    ap.add_argument("--ref-blocks", type=int, default=6, help="output blocks in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
