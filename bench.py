#!/usr/bin/env python
"""bench.py -- the pp-ladder hot path on B200: seconds per ppl_apply call and FP64 TFLOP/s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config large|xl|medium|small|tiny | --shape o,v,x]
                  [--impl ours|reference]

A "step" is one ppl_apply: the whole hot path (step 0 W-tile generation, step 1
(c,d) contraction, reduce/accumulate/mirror, ring/streams) over one seeded synthetic batch shaped
like BASELINE.json's configs.  Default workload: 'xl' (configs[4], the largest single-GPU config);
the default line also carries complete sub-records "large", "medium", "small", "tiny" (all five
configs of BASELINE.json; the launch-bound ones averaged over >= 50 calls).

value  = FP64 TFLOP/s on the USEFUL flops: what the exploited symmetry leaves of the nominal
         2*nchol*nvirt^4 + 2*nocc^2*nvirt^4 (ppl_info_t.flops_useful: no tile padding, no zero
         rows, no slab overshoot), inputs resident in HBM.  tflops_executed (the GEMM extents
         actually launched / time) is the kernel-efficiency figure beside it.
e2e    = the same through ppl_apply_host with pinned HOST buffers (H2D of L, t2, R and D2H of R
         inside the timed region).
roofline = the dominant kernel against the FP64 tensor (DMMA) pipe peak measured live by
         ppl_probe_fp64_peak (MEASURED_PEAKS.json carries no FP64 figure).
cpu_baseline = the oracle (oracle/ppl_oracle.c, as it stands) on the host cores, on a bounded
         sample of (a,b) columns of the same workload; the same sample is compared with the GPU
         result ("parity" key).
Multi-GPU: the path does not shard (north_star: one GPU, no collectives) -> "replicas only": under
torchrun every rank runs an independent replica; value is the aggregate, time the max over ranks.
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

# Headline: FP64 TFLOP/s on the flops the exploited symmetry leaves ("halved where symmetry is exploited, and stated",
# north_star) -- the symmetry-unique count flops_useful of ppl_info_t, with no tile padding, no zero rows and no
# slab-granularity overshoot in the numerator.  The rate on the GEMM extents actually launched
# (tflops_executed) is the kernel-efficiency number and stays in the line and in `roofline.achieved`.
METRIC = "pp_ladder_fp64_tflops_useful"
UNIT = "TFLOP/s"
SYM_NAMES = {0: "none", 1: "pair", 2: "pair_sa", 3: "full"}
SYM_DESC = {0: "none (every tile)", 1: "pair (tiles a-block<=b-block, mirrored)",
            2: "pair_sa (tiles a-block<=b-block, mirrored; step 1 on symmetric/antisymmetric packed (i<=j),(c<=d) operands: "
               "step-0 flops x~1/2, step-1 flops x~1/4 of nominal)",
            3: "full (8-fold ERI symmetry L[P,a,c]=L[P,c,a] + pair symmetry of t2: slabs of 16 a's, symmetric packed "
               "S+-[(a<=b)][(c<=d)] blocks generated once and used twice: step-0 flops x~1/8, step-1 flops x~1/4 of nominal)"}
NOMINAL_FP64_TFLOPS = 148 * 4 * 16 * 2 * 1.965e9 * 1e-12  # 148 SM x 4 SMSP x 16 FMA/clk x 2 x 1.965 GHz = 37.23


def col_flops(o, v, x):
    """flops of one (a,b) column of the two-step route: step 0 (2 x v^2) + step 1 (2 o^2 v^2)."""
    return 2.0 * x * v * v + 2.0 * o * o * v * v


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.proc:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        try:
            rows = [r.split(",") for r in open(self.path).read().strip().splitlines() if r.strip()]
            os.unlink(self.path)
        except Exception:
            return out
        sm, reasons = [], set()
        for r in rows:
            try:
                sm.append(float(r[0]))
                out["sm_max_mhz"] = float(r[1])
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if "Active" in val and "Not" not in val:
                        reasons.add(name)
            except Exception:
                continue
        if sm:
            sm.sort()
            out["sm_mhz"] = sm[len(sm) // 2]
            out["power_w_max"] = max(float(r[2]) for r in rows if len(r) > 2)
        out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


# --------------------------------------------------------------------------------------- reference
def oracle_sample(L, t2, o, v, x, target_s=15.0, seed=0):
    """Time oracle.columns on a bounded sample of (a,b) columns (~target_s of CPU work)."""
    import oracle
    import ppl_inputs as I

    pilot = I.sample_pairs(v, 4, seed=seed + 1)[:8]
    t0 = time.perf_counter()
    oracle.columns(L, t2, pilot)
    dt = max(time.perf_counter() - t0, 1e-4)
    per_col = dt / len(pilot)
    k = int(max(8, min(v * v, target_s / per_col)))
    pairs = I.sample_pairs(v, k, seed=seed)[:k]
    t0 = time.perf_counter()
    cols = oracle.columns(L, t2, pairs)
    dt = time.perf_counter() - t0
    return pairs, cols, dt, oracle.num_threads()


def run_reference(args, o, v, x):
    """--impl reference: the oracle as it stands on the host cores; each step = a bounded sample."""
    import ppl_inputs as I

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    L, t2 = I.make_L(v, x, 0), I.make_t2(o, v, 0)
    import oracle

    per_step_s = 8.0
    pilot = I.sample_pairs(v, 4, seed=1)[:8]
    t0 = time.perf_counter()
    oracle.columns(L, t2, pilot)
    per_col = max(time.perf_counter() - t0, 1e-4) / len(pilot)
    k = int(max(4, min(v * v, per_step_s / per_col)))
    pairs = I.sample_pairs(v, k, seed=0)[:k]
    for _ in range(args.warmup):
        oracle.columns(L, t2, pairs[: max(4, k // 8)])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.columns(L, t2, pairs)
    dt = time.perf_counter() - t0
    tflops = args.steps * len(pairs) * col_flops(o, v, x) / dt * 1e-12
    line = {
        "impl": "reference", "metric": METRIC, "value": tflops, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.config, o, v, x),
        "value_counts": "the oracle's own flops / time: it uses no symmetry, so this is the nominal count per (a,b) column; our arm "
                        "counts the symmetry-unique flops (1/5 of nominal at xl) -- for seconds per call compare seconds_per_call",
        "seconds_per_call": dt / args.steps / len(pairs) * v * v,
        "seconds_per_call_how": "EXTRAPOLATED: measured seconds per sampled (a,b) column x nvirt^2 columns",
        "cpu_baseline": {"value": tflops, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": f"{len(pairs)} of {v*v} (a,b) columns per step (oracle.columns), all i,j",
                         "extrapolated_seconds_per_call": dt / args.steps / len(pairs) * v * v},
        "e2e": {"value": tflops, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------- the paper's own Table 3 shapes (host-resident)
# Seconds per contraction printed in Table 3 for these shapes:
# operands in HOST memory, time includes batching, transfers and DGEMMs -- the same boundary as ppl_apply_host.
TABLE3_PAPER_SECONDS = {
    "table3_n800_o100": {"GH200 PyTorch C-split": 355.9, "GH200 CuPy C-split": 306.6, "H100 PyTorch C-split": 330.5,
                         "H100 CuPy C-split": 461.5, "GH200 PyTorch X-split": 574.7, "H100 PyTorch X-split": 789.4},
    "table3_n900_o100": {"GH200 PyTorch C-split": 587.1, "GH200 CuPy C-split": 495.0, "H100 PyTorch C-split": 496.2,
                         "H100 CuPy C-split": 809.7, "GH200 PyTorch X-split": 1265.7, "H100 PyTorch X-split": 1753.3},
    "table3_n800_o150": {"GH200 PyTorch C-split": 475.3, "GH200 CuPy C-split": 532.8, "H100 PyTorch C-split": 651.2,
                         "H100 CuPy C-split": 940.9, "GH200 PyTorch X-split": 637.4},
    "table3_n1000_o100": {"GH200 PyTorch C-split": 805.8, "GH200 CuPy C-split": 829.1, "H100 PyTorch C-split": 827.1,
                          "H100 CuPy C-split": 1338.7, "GH200 PyTorch X-split": 2673.7},
    "table3_n1000_o50": {"GH200 PyTorch C-split": 574.6, "GH200 CuPy C-split": 763.0, "H100 PyTorch C-split": 673.0,
                         "H100 CuPy C-split": 1006.4, "GH200 PyTorch X-split": 5262.6},
}


def run_table3(args, o, v, x):
    """--config table3_*: one of the paper's own benchmark shapes with HOST-resident operands.
    t2 and R (39 GB each at N=800, nocc=100) do not fit in HBM next to the workspace: ppl_apply_host streams them
    through staging buffers (PPL_SYM_FULL).  The only number is end to end: wall clock around ppl_apply_host."""
    import numpy as np
    import torch

    import paper_2603_20912_b200 as P
    import ppl_inputs as I

    if args.impl == "reference":
        print(json.dumps({"impl": "reference", "unavailable": "table3_* shapes are an e2e-only context workload; "
                          "the reference arm runs on the BASELINE.json configs"}))
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU path)")
    torch.cuda.set_device(0)
    t0 = time.perf_counter()
    # before anything else is allocated; the cap leaves room for what ppl_apply_host allocates on first use
    # (L whole + two 1-GiB staging buffers)
    free_b = torch.cuda.mem_get_info()[0]
    unpacked = args.symmetry in ("none", "pair")
    if unpacked:
        # the paper's own setting (unstructured random arrays, no symmetry used): nothing assumed of L, and
        # with `none` nothing of t2.  The plan needs only the W ring and the split-K partials; ppl_apply_host keeps t2
        # resident and streams L panels / R slabs beside it.
        cap = 8 << 30
    else:
        # room for what ppl_apply_host allocates on first use: L whole, two 1-GiB staging buffers, two R slabs of 16 a's
        cap = int(free_b * 0.98) - x * v * v * 8 - (2 << 30) - 2 * o * o * 16 * v * 8 - (1 << 30)
    plan = P.Plan(o, v, x, cap, debug={"host_panels": args.host_panels} if unpacked else None)
    if unpacked:
        plan.set_symmetry(P.PPL_SYM_NONE if args.symmetry == "none" else P.PPL_SYM_PAIR)
    plan_s = time.perf_counter() - t0
    info = plan.info()
    need = (x * v * v + 2 * o * o * v * v) * 8
    avail = 0
    for ln in open("/proc/meminfo"):
        if ln.startswith("MemAvailable"):
            avail = int(ln.split()[1]) * 1024
    if need > 0.845 * avail:  # pinned pages cannot be swapped; 162 GB of 194 GB pins on this pool's hosts, 166 GB does not
        plan.destroy()
        print(json.dumps({"unavailable": f"{need / 1e9:.0f} GB of pinned host operands on a host with {avail / 1e9:.0f} GB available"}))
        return
    t_gen = time.perf_counter()
    Lh = torch.empty((x, v, v), dtype=torch.float64, pin_memory=True)
    th = torch.empty((o, o, v, v), dtype=torch.float64, pin_memory=True)
    Rh = torch.zeros((o, o, v, v), dtype=torch.float64, pin_memory=True)
    I.make_L(v, x, 0, symmetric=not unpacked, out=Lh.numpy())
    I.make_t2(o, v, 0, symmetric=args.symmetry != "none", out=th.numpy())
    t_gen = time.perf_counter() - t_gen
    sampler = ClockSampler(0)
    for _ in range(max(args.warmup, 0)):
        plan.apply_host(Lh, th, Rh)
    Rh.zero_()
    sampler.start()
    secs = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        h2d, d2h = plan.apply_host(Lh, th, Rh)
        secs.append(time.perf_counter() - t0)
    clocks = sampler.stop()
    dt = sum(secs) / len(secs)
    f_exec, f_nom = info["flops_executed"], info["flops_nominal"]
    paper = TABLE3_PAPER_SECONDS.get(args.config, {})
    best = min(paper.values()) if paper else None
    line = {
        "metric": "pp_ladder_seconds_per_call_host_resident", "value": dt, "unit": "s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": (dt / best) if best else None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.config, "nocc": o, "nvirt": v, "nchol": x, "seed": 0,
                   "note": "shape of the paper's Table 3 row (PAPER.md:417-451); operands in pinned HOST memory; " +
                           ({"none": "UNSTRUCTURED L and t2 (no symmetry generated, none assumed or used: the paper's own "
                                     "setting, PAPER.md:385); t2 resident, L whole or in row panels, R in slabs",
                             "pair": "unstructured L, pair-symmetric t2; t2 and R resident, L whole or in row panels"}.get(
                                 args.symmetry, "symmetric L and pair-symmetric t2 (the paper used unstructured random "
                                                "arrays and no symmetry)")),
                   "host_panels": args.host_panels if unpacked else None,
                   "symmetry": SYM_DESC[info["symmetry"]],
                   "plan": {k: info[k] for k in ("ta", "tb", "n_tiles", "workspace_bytes", "full_tight")}},
        "step_seconds": secs, "plan_seconds": plan_s, "input_gen_seconds": t_gen,
        "tflops_executed": f_exec / dt * 1e-12, "tflops_nominal_effective": f_nom / dt * 1e-12,
        "flops_executed": f_exec, "flops_nominal": f_nom,
        "e2e": {"value": dt, "unit": "s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "how": "ppl_apply_host on pinned host buffers; wall clock around the synchronous call"},
        "paper_seconds_other_hardware": paper, "clocks": clocks,
        "gpu_launches": info["launches_per_apply"] * args.steps,
    }
    if not args.no_cpu_baseline:
        Rh.zero_()
        plan.apply_host(Lh, th, Rh)  # exactly one application of the term for the comparison
        pairs, cols, dto, cores = oracle_sample(Lh.numpy(), th.numpy(), o, v, x, target_s=20.0)
        got = Rh.numpy()[:, :, pairs[:, 0], pairs[:, 1]].transpose(2, 0, 1)
        err = float(np.abs(got - cols).max() / np.abs(cols).max())
        line["cpu_baseline"] = {"value": dto / len(pairs) * v * v, "unit": "s (extrapolated from the sample)", "cores": cores,
                                "kind": "oracle", "sample": f"{len(pairs)} of {v*v} (a,b) columns (oracle.columns), all i,j; {dto:.1f} s"}
        line["parity"] = {"max_rel_err_vs_oracle": err, "tolerance": 1e-11, "columns": int(len(pairs)), "ok": bool(err <= 1e-11)}
    plan.destroy()
    print(json.dumps(line))


# ------------------------------------------------------------------------------ N > 1: replicas only
def paper_recipe_leg(Ld, td, Rd_ours, steps: int, w_bytes: float = 8e9) -> dict:
    """CONTEXT ONLY (optional row): the paper's own recipe re-expressed on this B200 with library calls.

    PAPER.md:146-181 (C-split): for b-chunks, for a-chunks: `result_temp = tensordot(chol_1[a], chol_2, axes=(0, 0))`
    ('xac,xbd->acbd'), `result_temp_2 = tensordot(result_temp, operand2, axes=([1, 3], [c, d]))`
    ('acbd,ecfd->abef', :171-173), transpose, add to the view of the result (:175-177).  Here in the setting most
    favourable to it: all operands already resident in HBM (no host<->device traffic, n_c = 1), square (a, b) chunks
    sized so that result_temp plus the permuted copy tensordot makes of it fit in `w_bytes`, PyTorch FP64 tensordot =
    cuBLAS DGEMM.  No symmetry (the paper exploits none on this path).  None of this repo's kernels run here.
    """
    import torch

    x, v, _ = Ld.shape
    o = td.shape[0]
    n = max(1, min(v, int((w_bytes / (2 * 8 * v * v)) ** 0.5)))
    R = torch.zeros_like(Rd_ours)

    def one():
        for b0 in range(0, v, n):
            chol_2 = Ld[:, b0:b0 + n, :]
            for a0 in range(0, v, n):
                chol_1 = Ld[:, a0:a0 + n, :]
                result_temp = torch.tensordot(chol_1, chol_2, dims=([0], [0]))          # [a, c, b, d]
                result_temp_2 = torch.tensordot(result_temp, td, dims=([1, 3], [2, 3]))  # [a, b, i, j]
                del result_temp
                R[:, :, a0:a0 + n, b0:b0 + n] += result_temp_2.permute(2, 3, 0, 1)
                del result_temp_2

    one()  # warm-up (cuBLAS handles, allocator)
    torch.cuda.synchronize()
    diff = float((R - Rd_ours).abs().max() / Rd_ours.abs().max())
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(steps):
        one()
    ev1.record()
    torch.cuda.synchronize()
    dt = ev0.elapsed_time(ev1) * 1e-3 / steps
    f_nom = 2.0 * x * v ** 4 + 2.0 * o * o * v ** 4
    del R
    torch.cuda.empty_cache()
    return {"seconds_per_call": dt, "tflops_nominal": f_nom / dt * 1e-12, "steps": steps, "chunk_a": n, "chunk_b": n,
            "max_rel_diff_vs_ours": diff,
            "what": "the paper's C-split recipe (PAPER.md:146-181) as two torch.tensordot calls (cuBLAS DGEMM) per "
                    "(a, b) chunk + transpose + add, operands resident in HBM, no symmetry; context, not the product"}


def max_over_ranks(ms: float, dist, device) -> float:
    """Device time of the slowest rank (one scalar all-reduce: plumbing, not data path). dist=None: one process."""
    if dist is None:
        return ms
    import torch

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_value(flops_per_replica: float, ms_per_step: float, world: int) -> float:
    """Whole-job TFLOP/s of `world` independent replicas that all finished within ms_per_step (the max over ranks)."""
    return world * flops_per_replica / (ms_per_step * 1e-3) * 1e-12


# -------------------------------------------------------------------------------------------- ours
L2_BYTES = 126 << 20


def workload_config(name, o, v, x):
    """The `config` object: identical in both arms (ours / reference) so that the lines are comparable."""
    small = (x * v * v + 2 * o * o * v * v) * 8 < 2 * L2_BYTES
    return {"workload": name, "nocc": o, "nvirt": v, "nchol": x, "seed": 0,
            "l2": ("flushed between timed iterations (256 MiB memset outside the event pair): inputs smaller than L2"
                   if small else "inputs larger than L2 (L, t2, W tiles >> 126 MB); no flush needed")}


def probe_leg():
    """--probe: the instruction streams the pipe choice was made between, cuBLAS DGEMM for context, clocks."""
    import torch

    import paper_2603_20912_b200 as P

    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    sampler.start()
    out = {k: P.ppl_probe_fp64_pipe(k, 3, 50.0) for k in ("dmma8", "dmma16", "dfma16", "mix8")}
    n = 8192
    a = torch.randn(n, n, dtype=torch.float64, device="cuda")
    b = torch.randn(n, n, dtype=torch.float64, device="cuda")
    for _ in range(2):
        torch.matmul(a, b)
    best = 0.0
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, 2.0 * n ** 3 / (e0.elapsed_time(e1) * 1e-3) * 1e-12)
    out["cublas_dgemm_8192"] = best
    out["nominal"] = NOMINAL_FP64_TFLOPS
    out["unit"] = UNIT
    out["clocks"] = sampler.stop()
    out["what"] = ("register-only loops, 16 warps/SM x 148 SMs: dmma8/dmma16 = mma.sync.m8n8k4.f64 with 8/16 independent "
                   "accumulator chains per warp; dfma16 = DFMA, 16 chains per thread; mix8 = DMMA + DFMA interleaved "
                   "(flops of both counted); cublas = torch.matmul FP64 8192^3 best of 10 (library bar, context)")
    print(json.dumps(out))


def contract_leg():
    """--contract: ppl_contract_pair (the generic 'op0,op1->out' entry point) on the paper's two ladder
    strings at slab sizes of the medium / large configs, with torch.einsum (cuBLAS + permuted copies: the paper's
    tensordot route on this box) beside it as context."""
    import torch

    import paper_2603_20912_b200 as P

    torch.cuda.set_device(0)
    peak = P.ppl_probe_fp64_peak(3, 20.0)
    out = {"peak": peak, "unit": UNIT, "cases": []}
    cases = [
        ("xac,xbd->acbd", (800, 16, 200), (800, 200, 200)),      # step 0, one slab of 16 a's at medium
        ("abcd,efcd->efab", (16, 200, 200, 200), (20, 20, 200, 200)),  # step 1 on that slab, t2 stored [i,j,c,d]
        ("abcd,ecfd->efab", (16, 200, 200, 200), (20, 200, 20, 200)),  # the paper's own string: t2 stored [i,c,j,d]
        ("xac,xbd->acbd", (1600, 4, 400), (1600, 400, 400)),     # step 0, 4 a's at large (output 2 GB)
        ("abcd,ecfd->efab", (4, 400, 400, 400), (40, 400, 40, 400)),
        ("ik,kj->ij", (4096, 4096), (4096, 4096)),
    ]
    for subs, sa, sb in cases:
        g = torch.Generator(device="cuda").manual_seed(0)
        A = torch.randn(sa, dtype=torch.float64, device="cuda", generator=g)
        B = torch.randn(sb, dtype=torch.float64, device="cuda", generator=g)
        C = P.ppl_contract_pair(subs, A, B)
        torch.cuda.synchronize()
        ref = torch.einsum(subs, A, B)
        err = float((C - ref).abs().max() / ref.abs().max())
        ins, _ = subs.split("->")
        s0, s1 = ins.split(",")
        ext = dict(zip(s0, sa))
        ext.update(zip(s1, sb))
        flops = 2.0
        for val in ext.values():
            flops *= val
        res = {}
        for name, fn in (("ours", lambda: P.ppl_contract_pair(subs, A, B, C)), ("torch_einsum", lambda: torch.einsum(subs, A, B))):
            for _ in range(2):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                fn()
            e1.record()
            torch.cuda.synchronize()
            res[name] = flops / (e0.elapsed_time(e1) / 5 * 1e-3) * 1e-12
        out["cases"].append({"subscripts": subs, "dims0": sa, "dims1": sb, "flops": flops, "tflops": res["ours"],
                             "frac_of_peak": res["ours"] / peak, "torch_einsum_tflops": res["torch_einsum"],
                             "max_rel_diff_vs_torch": err})
        del A, B, C, ref
        torch.cuda.empty_cache()
    print(json.dumps(out))


def entry_points_leg(peak, plain_seconds):
    """The widened entry points at `large`: seconds and TFLOP/s of ppl_apply_ex in the paper's storage
    orders ('icjd' -> 'iajb', alpha != 1, beta = 0; the permutation is folded into the pack / unpack kernels),
    of ppl_generate_eri + ppl_apply_dense on one slab of 16 a's, and of ppl_contract_pair on the ladder's strings."""
    import torch

    import paper_2603_20912_b200 as P
    import ppl_inputs as I

    o, v, x = I.CONFIGS["large"]
    Ld = torch.from_numpy(I.make_L(v, x, 0)).cuda()
    td = torch.from_numpy(I.make_t2(o, v, 0)).cuda()
    t_icjd = td.permute(0, 2, 1, 3).contiguous()
    R_iajb = torch.empty((o, v, o, v), dtype=torch.float64, device="cuda")
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")

    def timed(fn, n=3, warm=1):
        for _ in range(warm):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e-3

    out = {"workload": "large", "peak": peak, "unit": UNIT}
    with P.Plan(o, v, x) as plan:
        info = plan.info()
        t_ex = timed(lambda: plan.apply_ex(Ld, t_icjd, R_iajb, "iajb", "iajb", alpha=-0.625, beta=0.0))
        out["apply_ex_iajb_beta0"] = {"seconds_per_call": t_ex, "plain_apply_seconds": plain_seconds,
                                      "over_plain": t_ex / plain_seconds if plain_seconds else None,
                                      "tflops_executed": info["flops_executed"] / t_ex * 1e-12,
                                      "frac_of_peak": info["flops_executed"] / t_ex * 1e-12 / peak}
        na = 16
        eri = torch.empty((na, v, v, v), dtype=torch.float64, device="cuda")
        t_gen = timed(lambda: plan.generate_eri(Ld, 64, na, eri))
        f_gen = 2.0 * x * na * v ** 3
        out["generate_eri_16"] = {"seconds_per_call": t_gen, "tflops": f_gen / t_gen * 1e-12, "frac_of_peak": f_gen / t_gen * 1e-12 / peak}
        t_dense = timed(lambda: plan.apply_dense(eri, 64, td, Rd))
        f_dense = 2.0 * o * o * na * v ** 3
        out["apply_dense_16"] = {"seconds_per_call": t_dense, "tflops": f_dense / t_dense * 1e-12,
                                 "frac_of_peak": f_dense / t_dense * 1e-12 / peak}
        del eri
    del Rd, R_iajb, t_icjd
    torch.cuda.empty_cache()
    out["contract_pair"] = []
    for subs, A, B in (("xac,xbd->acbd", Ld[:, 200:204, :].contiguous(), Ld),
                       ("abcd,ecfd->efab", torch.randn((4, v, v, v), dtype=torch.float64, device="cuda"), td.permute(0, 2, 1, 3).contiguous()),
                       ("ik,kj->ij", torch.randn((4096, 4096), dtype=torch.float64, device="cuda"),
                        torch.randn((4096, 4096), dtype=torch.float64, device="cuda"))):
        C = P.ppl_contract_pair(subs, A, B)
        ins, _ = subs.split("->")
        s0, s1 = ins.split(",")
        ext = dict(zip(s0, A.shape))
        ext.update(zip(s1, B.shape))
        flops = 2.0
        for val in ext.values():
            flops *= val
        t = timed(lambda: P.ppl_contract_pair(subs, A, B, C), n=5, warm=2)
        out["contract_pair"].append({"subscripts": subs, "dims0": list(A.shape), "dims1": list(B.shape), "seconds_per_call": t,
                                     "tflops": flops / t * 1e-12, "frac_of_peak": flops / t * 1e-12 / peak})
        del A, B, C
    torch.cuda.empty_cache()
    return out


def run_ours(name, o, v, x, args, steps, warmup, dist, dev, rank, world, peak):
    """One workload through ppl_apply (device-resident), ppl_apply_profiled (roofline), ppl_apply_host (e2e) and the
    oracle sample (cpu_baseline + parity).  Returns the JSON record."""
    import numpy as np
    import torch

    import paper_2603_20912_b200 as P
    import ppl_inputs as I

    # ---- seeded synthetic inputs in pinned host memory (shared bit-for-bit with the oracle) ----
    t_gen = time.perf_counter()
    Lh = torch.empty((x, v, v), dtype=torch.float64, pin_memory=True)
    th = torch.empty((o, o, v, v), dtype=torch.float64, pin_memory=True)
    Rh = torch.zeros((o, o, v, v), dtype=torch.float64, pin_memory=True)
    I.make_L(v, x, 0, out=Lh.numpy())
    I.make_t2(o, v, 0, out=th.numpy())
    t_gen = time.perf_counter() - t_gen
    Ld, td = Lh.to(dev, non_blocking=True), th.to(dev, non_blocking=True)
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device=dev)
    torch.cuda.synchronize()

    t0 = time.perf_counter()
    debug = {"no_small_fused": 1} if args.no_small_fused else {}
    for kv in (args.debug.split(",") if args.debug else []):  # A/B runs: ppl_debug_opts_t fields by name
        k_, v_ = kv.split("=")
        debug[k_] = int(v_)
    plan = P.Plan(o, v, x, int(args.workspace_gb * (1 << 30)), debug=debug or None)
    plan_s = time.perf_counter() - t0
    if args.symmetry != "default":
        plan.set_symmetry({v_: k_ for k_, v_ in SYM_NAMES.items()}[args.symmetry])
    plan.set_graph({"auto": -1, "off": 0, "on": 1}[args.graph])
    if args.verify >= 0:
        plan.set_verify(args.verify)
    info = plan.info()
    stream = torch.cuda.current_stream()
    cfg = workload_config(name, o, v, x)
    flush = cfg["l2"].startswith("flushed")
    scratch = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if flush else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(warmup, 0)):
        plan.apply(Ld, td, Rd)
    barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    barrier()
    for k in range(steps):
        if flush:
            scratch.zero_()  # outside the event pair
        ev0[k].record(stream)
        plan.apply(Ld, td, Rd)  # R accumulates (+=) across steps; no work is skipped
        ev1[k].record(stream)
    barrier()
    clocks = sampler.stop()
    step_ms = [ev0[k].elapsed_time(ev1[k]) for k in range(steps)]
    # without a flush the steps run back to back: the span first start -> last end is the timed region
    total_ms = sum(step_ms) if flush else ev0[0].elapsed_time(ev1[-1])
    total_ms = max_over_ranks(total_ms, dist, dev)
    ms_per_step = total_ms / steps
    sec = ms_per_step * 1e-3
    f_exec, f_nom, f_use = info["flops_executed"], info["flops_nominal"], info["flops_useful"]
    value = replicas_value(f_use, ms_per_step, world)

    # ---- dominant kernel, timed live with CUDA events on the launching stream (serialised pass) ----
    Rd.zero_()
    prof = plan.apply_profiled(Ld, td, Rd)  # Rd now holds exactly one application of the term
    torch.cuda.synchronize()
    dom = "step0" if prof["step0_ms"] >= prof["step1_ms"] else "step1"
    fused = bool(info.get("small_fused"))
    # the one-kernel path of launch-bound shapes does both steps in its single launch (timed as "step0")
    dom_total = info["flops_executed"] if fused else info["flops_" + dom]
    dom_flops = dom_total / max(prof["n_" + dom], 1)
    dom_ms = prof[dom + "_ms"] / max(prof["n_" + dom], 1)
    achieved = dom_flops / (dom_ms * 1e-3) * 1e-12
    dom_useful = (info["flops_useful"] if fused else info["flops_useful_" + dom]) / (prof[dom + "_ms"] * 1e-3) * 1e-12
    traffic = None
    try:
        import csv

        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "dram_traffic.csv"))):
            if row["config"] == name and row["symmetry"] == SYM_NAMES[info["symmetry"]] and row["kernel"] == dom:
                traffic = float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    roofline = {
        "bound": "tensor", "kernel": "k_small_fused" if fused else "k_" + dom, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
        "frac": achieved / peak, "traffic": traffic,
        "achieved_useful": dom_useful, "frac_useful": dom_useful / peak,
        "peak_source": "measured live: ppl_probe_fp64_peak (register-only DMMA m8n8k4 stream; profiles/r02_fp64_peaks.md); "
                       f"nominal {NOMINAL_FP64_TFLOPS:.2f} = 148 SM x 4 SMSP x 16 FMA/clk x 2 x 1.965 GHz",
        "flops_per_launch": dom_flops, "ms_per_launch": dom_ms,
        "how": "ppl_apply_profiled: one serialised apply after the timed steps, a CUDA event pair around every launch; "
               "achieved = flops of the GEMM extents launched / time, achieved_useful = the symmetry-unique flops of the "
               "same launches / the same time",
        "step0_tflops": info["flops_step0"] / (prof["step0_ms"] * 1e-3) * 1e-12 if prof["step0_ms"] > 0 else None,
        "step1_tflops": info["flops_step1"] / (prof["step1_ms"] * 1e-3) * 1e-12 if prof["step1_ms"] > 0 else None,
        "share": {"step0": prof["step0_ms"] / prof["total_ms"], "step1": prof["step1_ms"] / prof["total_ms"],
                  "reduce": prof["reduce_ms"] / prof["total_ms"], "fold": prof["fold_ms"] / prof["total_ms"],
                  "pack": prof["pack_ms"] / prof["total_ms"]},
        "launches": {k: prof["n_" + k] for k in ("step0", "step1", "reduce", "fold", "pack")},
    }
    if fused:
        # launch-bound shapes: one fused launch; the FP64 pipe is not what bounds it (profiles/r02_small_fused.md)
        roofline["limiter"] = ("launch + shared-memory latency, not the tensor pipe: one launch per apply (floor 4-5 us); at "
                               "`small` the work decomposition (one warp = one (a,b) column, t2 re-read from shared memory per "
                               "column) has a floor of about 100 us")

    rec = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": cfg,
        "value_counts": "flops_useful (symmetry-unique flops of the mode: no tile padding, no zero rows, no slab overshoot) / "
                        "time; tflops_executed counts the GEMM extents launched",
        "run": {"symmetry": SYM_DESC[info["symmetry"]], "parallelism": "replicas only" if world > 1 else "1 gpu",
                "plan": {k: info[k] for k in ("ta", "tb", "n_tiles", "ring", "splitk", "vec16", "workspace_bytes")},
                "graph": args.graph, "verify_inputs": 1 if args.verify < 0 else args.verify, "small_fused": info.get("small_fused", 0)},
        "seconds_per_call": sec,
        "tflops_executed": f_exec / sec * 1e-12,
        "tflops_useful": f_use / sec * 1e-12,
        "tflops_nominal_effective": f_nom / sec * 1e-12,
        "flops_executed": f_exec, "flops_useful": f_use, "flops_nominal": f_nom,
        "executed_over_useful": f_exec / f_use,
        "frac_of_fp64_peak_measured": f_exec / sec * 1e-12 / peak,
        "frac_of_fp64_peak_measured_useful": f_use / sec * 1e-12 / peak,
        "frac_of_fp64_peak_nominal": f_exec / sec * 1e-12 / NOMINAL_FP64_TFLOPS,
        "step_ms": step_ms, "plan_seconds": plan_s, "input_gen_seconds": t_gen,
        "clocks": clocks, "roofline": roofline,
        "gpu_launches": info["launches_per_apply"] * steps,
    }

    if rank == 0 and not args.no_e2e:
        # ---- end to end through the host entry point: H2D(L, t2, R) + apply + D2H(R) per step ----
        n_e2e = max(1, args.e2e_steps if args.e2e_steps > 0 else steps)
        Rh.zero_()
        h2d, d2h = plan.apply_host(Lh, th, Rh)  # warm-up (allocates the staging buffers)
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            h2d, d2h = plan.apply_host(Lh, th, Rh)
        dt = (time.perf_counter() - t0) / n_e2e
        rec["e2e"] = {"value": world * f_use / dt * 1e-12, "unit": UNIT, "h2d_bytes_per_step": h2d,
                      "d2h_bytes_per_step": d2h, "seconds_per_call": dt, "steps": n_e2e,
                      "tflops_executed": world * f_exec / dt * 1e-12,
                      "how": "ppl_apply_host on pinned host buffers; wall clock around the synchronous call"}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # ---- the oracle on the host cores, bounded sample; the same sample checks the GPU result ----
        pairs, cols, dt, cores = oracle_sample(Lh.numpy(), th.numpy(), o, v, x, target_s=getattr(args, "oracle_target_s", 15.0))
        rec["cpu_baseline"] = {
            "value": len(pairs) * col_flops(o, v, x) / dt * 1e-12, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{len(pairs)} of {v*v} (a,b) columns (oracle.columns), all i,j; {dt:.1f} s",
            "extrapolated_seconds_per_call": dt / len(pairs) * v * v,
        }
        Rg = Rd.cpu().numpy()
        got = Rg[:, :, pairs[:, 0], pairs[:, 1]].transpose(2, 0, 1)
        err = float(np.abs(got - cols).max() / np.abs(cols).max())
        rec["parity"] = {"max_rel_err_vs_oracle": err, "tolerance": 1e-11, "columns": int(len(pairs)), "ok": bool(err <= 1e-11)}

    if rank == 0 and world == 1 and args.paper_recipe > 0:
        Rd.zero_()
        plan.apply(Ld, td, Rd)
        torch.cuda.synchronize()
        rec["paper_recipe"] = paper_recipe_leg(Ld, td, Rd, args.paper_recipe)

    plan.destroy()
    del Ld, td, Rd, Lh, th, Rh, scratch
    torch.cuda.empty_cache()
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="xl", help="xl (default: the largest single-GPU config of BASELINE.json; the line "
                    "then also carries a complete 'large' record), large, medium, small, tiny, table3_*")
    ap.add_argument("--shape", default=None, help="nocc,nvirt,nchol: a custom shape with the same generators (overrides --config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workspace-gb", type=float, default=0.0, help="workspace cap (0 = auto)")
    ap.add_argument("--symmetry", default="default", choices=["default", "full", "pair_sa", "pair", "none"],
                    help="default = the plan's own choice (full: 8-fold ERI symmetry + pair symmetry, from nvirt = 52 up)")
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="ppl_plan_set_graph: replay one CUDA graph per apply (auto: launch-bound shapes only)")
    ap.add_argument("--verify", type=int, default=-1, choices=[-1, 0, 1, 2],
                    help="PPL_OPT_VERIFY_INPUTS (-1 = the library default: 1, a symmetry check at the head of every apply)")
    ap.add_argument("--no-small-fused", action="store_true",
                    help="A/B: send launch-bound shapes (tiny, small) through the tiled path instead of the one fused kernel")
    ap.add_argument("--host-panels", type=int, default=0, choices=[0, 1, 2],
                    help="table3_* with --symmetry none|pair: 1 = stream L as row panels even if it fits whole, 2 = never")
    ap.add_argument("--debug", default="", help="ppl_debug_opts_t fields for A/B runs, e.g. full_group_m=12,full_hints=5")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=0, help="timed ppl_apply_host calls (0 = --steps)")
    ap.add_argument("--no-secondary", action="store_true", help="with --config xl: skip the 'large' sub-record")
    ap.add_argument("--paper-recipe", type=int, default=0, metavar="STEPS",
                    help="context leg: time STEPS calls of the paper's tensordot recipe (cuBLAS) on the same inputs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--contract", action="store_true", help="only time ppl_contract_pair on the paper's two ladder strings")
    ap.add_argument("--sweep", action="store_true", help="molecule-like shapes between medium and large (Table 4 of the paper, "
                    "PAPER.md:466-507: odd nvirt, nvirt = 8 mod 16, ...): one compact record per shape in one JSON line")
    ap.add_argument("--entry-points", action="store_true", help="only the entry_points record (ppl_apply_ex in the paper's layouts, "
                    "ppl_generate_eri + ppl_apply_dense, ppl_contract_pair) at large")
    ap.add_argument("--probe", action="store_true", help="only measure the FP64 instruction-stream peaks and print them")
    args = ap.parse_args()

    import ppl_inputs as I

    if args.probe:
        probe_leg()
        return
    if args.contract:
        contract_leg()
        return
    if args.entry_points:
        import torch

        import paper_2603_20912_b200 as P

        torch.cuda.set_device(0)
        print(json.dumps(entry_points_leg(P.ppl_probe_fp64_peak(3, 20.0), None)))
        return
    if args.shape:
        o, v, x = (int(t) for t in args.shape.split(","))
        args.config = f"custom_{o}_{v}_{x}"
    elif args.config in I.TABLE3_SHAPES:
        run_table3(args, *I.TABLE3_SHAPES[args.config])
        return
    else:
        o, v, x = I.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, o, v, x)
        return

    import torch

    import paper_2603_20912_b200 as P

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU path)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    peak = P.ppl_probe_fp64_peak(3, 20.0)

    if args.sweep:
        # shapes of the medium class, where the paper's molecules live ((H2O)10 / cc-pVDZ is nocc 40, nvirt 190)
        shapes = [(20, 200, 800), (40, 190, 1150), (40, 191, 1150), (30, 230, 1200), (25, 260, 1300), (40, 264, 1400),
                  (32, 296, 1500), (48, 312, 1700), (64, 330, 1970), (36, 360, 1800), (40, 400, 1600), (40, 401, 1600),
                  (50, 450, 2200), (40, 530, 2850)]
        args.no_e2e, args.oracle_target_s = True, 4.0
        recs = []
        for (so, sv, sx) in shapes:
            r = run_ours(f"sweep_{so}_{sv}_{sx}", so, sv, sx, args, args.steps, args.warmup, dist, dev, rank, world, peak)
            recs.append({"shape": [so, sv, sx], "seconds_per_call": r["seconds_per_call"], "tflops_executed": r["tflops_executed"],
                         "tflops_useful": r["tflops_useful"], "frac_executed": r["frac_of_fp64_peak_measured"],
                         "frac_useful": r["frac_of_fp64_peak_measured_useful"], "executed_over_useful": r["executed_over_useful"],
                         "share": r["roofline"]["share"], "launches": r["roofline"]["launches"],
                         "step0_tflops": r["roofline"]["step0_tflops"], "step1_tflops": r["roofline"]["step1_tflops"],
                         "plan": r["run"]["plan"], "parity": r.get("parity"), "clocks": r["clocks"]})
        if rank == 0:
            print(json.dumps({"sweep": recs, "peak": peak, "unit": UNIT, "steps": args.steps, "warmup": args.warmup}))
        return
    line = run_ours(args.config, o, v, x, args, args.steps, args.warmup, dist, dev, rank, world, peak)
    if args.config == "xl" and not args.no_secondary and not args.shape:
        # BASELINE.json quotes the metric on "the two largest configs": the other one rides on the same line
        lo, lv, lx = I.CONFIGS["large"]
        line["large"] = run_ours("large", lo, lv, lx, args, args.steps, args.warmup, dist, dev, rank, world, peak)
        if rank == 0 and world == 1:
            line["entry_points"] = entry_points_leg(peak, line["large"]["seconds_per_call"])
        # ... and north_star asks for all five: medium, small and tiny as complete sub-records too (averaged over more
        # calls, the launch-bound ones over >= 50; they add about a minute, most of it the oracle samples)
        for name, nsteps in (("medium", max(args.steps, 20)), ("small", max(args.steps, 50)), ("tiny", max(args.steps, 50))):
            so, sv, sx = I.CONFIGS[name]
            line[name] = run_ours(name, so, sv, sx, args, nsteps, max(args.warmup, 5), dist, dev, rank, world, peak)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


if __name__ == "__main__":
    main()
