#!/usr/bin/env python
"""bench.py -- one JSON line per run (driver contract + tier framing).

A "step" = one pass of the WHOLE hot path over one tensor of the workload: fusefss_keygen (both key bundles),
fusefss_eval_cmp + fusefss_eval_lut for party 0 and party 1, fusefss_post_fused.  `value` = elements/s of that
whole step, inputs resident in HBM; eval-only and keygen-only rates, key and online bytes per element and the
roofline of the dominant kernel (k_gen_vec; k_eval_lut beside it) ride along, as do the same workload compiled with the
single-key shared-prefix construction (`shared_prefix`, `shared_prefix_public_horner`), the PRG / pipe probes and the
Eq. 1 LAN/WAN projection.  `e2e` = the same gate through fusefss_gate_host with
pinned HOST buffers (H2D + D2H inside the timed region).  `--impl reference` times the CPU oracle instead.
N > 1 (torchrun): every rank runs the full tensor on its own GPU (elements are independent gate instances,
no collective); value = N * count / max-over-ranks time; scaling = "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "compiled-op elements/s (keygen + cmp+LUT eval both parties + post); also eval-only and keygen-only elems/s; key B/elem"
SM_CLOCK_MAX_MHZ = 1965.0
LOOKUPS_PER_AES = 160           # 16 table lookups x 10 rounds (DESIGN 5.2)
# dram__bytes_read.sum + dram__bytes_write.sum per launch from `ncu --set full` (profiles/r1c_gelu.md)
NCU_TRAFFIC = {("gelu", 393216, "k_gen_vec"): 20.406e9, ("gelu", 393216, "k_eval_lut"): 10.279e9,
               ("gelu", 393216, "k_eval_sp"): 1.389e9}           # k_eval_sp<3,1>: profiles/r1h_gelu.md


def project(t_comp_ms, bytes_per_party, rounds):
    """Eq. 1 of the paper: T_proj = T_comp + 2 B_comm / BW + R RTT, with its LAN / WAN parameters."""
    return {"t_comp_ms": t_comp_ms, "bytes_per_party": bytes_per_party, "rounds": rounds,
            "lan_ms": t_comp_ms + 2e3 * bytes_per_party / 1e9 + rounds * 0.5,
            "wan_ms": t_comp_ms + 2e3 * bytes_per_party / 400e6 + rounds * 4.0}
LDS_LANES_PER_CLK_SM = 32       # shared-memory crossbar: 128 B/clk/SM (B300_MICROARCH "LDS/STS")


def aes_per_elem(shape, n):
    """AES blocks per element: (eval of ONE party, keygen of both bundles) -- DESIGN 5.3"""
    Q = (shape["p"] + 1) // 2
    ev = sum(k + 1 for k in shape["k"])
    gen = sum(4 * k + 2 + 2 for k in shape["k"])
    if shape["has_lut"]:
        ev += (shape["M"] - 1) * (n * (1 + Q) + Q)
        gen += (shape["M"] - 1) * (4 * n * (1 + Q) + 2 * Q + 2)
    return ev, gen


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.samples, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([v.strip() for v in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm = [float(s[0]) for s in self.samples if s and s[0].replace(".", "").isdigit()]
        reasons = set()
        for s in self.samples:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), s[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        mx = [float(s[1]) for s in self.samples if len(s) > 1 and s[1].replace(".", "").isdigit()]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(self.samples)}


def cpu_oracle_rate(name, sample, seed=0):
    """The oracle as it stands (single thread) on a bounded sample: whole gate (keygen + eval x2 + post)."""
    import oracle
    from workloads import specs, tensors
    spec = specs.CONFIGS[name]()
    O = oracle.Program(spec)
    inp = tensors.inputs(name, spec, count=sample, seed=seed)
    t0 = time.perf_counter()
    k0, k1 = O.keygen(inp["r_in"], inp["r_out"], seed)
    t1 = time.perf_counter()
    O.run_gate(k0, k1, inp["xhat"])
    t2 = time.perf_counter()
    return sample / (t2 - t0), dict(keygen_elems_per_s=sample / (t1 - t0), eval_post_elems_per_s=sample / (t2 - t1), seconds=t2 - t0)


def run_reference(args, rank):
    if rank != 0:
        return
    sample = args.ref_sample
    vals = []
    for i in range(args.warmup + args.steps):
        v, _ = cpu_oracle_rate(args.workload, sample, seed=i)
        if i >= args.warmup:
            vals.append((v, sample / v))
    value = sample * len(vals) / sum(t for _, t in vals)
    cores = 1
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "elements/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(t for _, t in vals) / len(vals),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": args.workload, "sample": f"first {sample} elements per step"},
            "cpu_baseline": {"value": value, "unit": "elements/s", "cores": cores, "kind": "oracle",
                             "sample": f"{sample} elements of {args.workload}, whole gate (keygen + eval both parties + post), single thread"},
            "e2e": {"value": value, "unit": "elements/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def measure_shared_prefix(F, torch, name, base_spec, inp, rank, world, steps, warmup, barrier, max_over_ranks, xpoly=False):
    """The same workload compiled with variant 1 (single-key shared-prefix construction):
    keygen (one n-bit key per element) + ONE fused evaluation per party + post, timed like the main step."""
    from workloads import specs as _specs
    spec = _specs.shared_prefix(base_spec)
    if xpoly:
        spec = _specs.public_point_horner(spec)
    P = F.Program(spec)
    sh, cost = P.shape, P.cost()
    count = int(inp["xhat"].size)
    torch.cuda.empty_cache()
    free_b, _ = torch.cuda.mem_get_info()
    if 2 * P.key_bytes(count) + 8 * count * (8 + 2 * sh["p"]) > 0.85 * free_b:
        return {"skipped": "variant-1 keys of the whole tensor do not fit resident"}
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    r_in, r_out, xhat = dev(inp["r_in"]), dev(inp["r_out"]), dev(inp["xhat"])
    k0, k1 = P.alloc_keys(count)
    na = max(1, sh["n_out_a"])
    bits = [torch.empty(count, dtype=torch.int64, device="cuda") for _ in (0, 1)]
    coeff = [torch.empty((sh["p"], count), dtype=torch.int64, device="cuda") for _ in (0, 1)]
    outs = (torch.empty((na, count), dtype=torch.int64, device="cuda"), torch.empty((na, count), dtype=torch.int64, device="cuda"),
            torch.empty(count, dtype=torch.int64, device="cuda"), torch.empty(count, dtype=torch.int64, device="cuda"))
    ev = lambda: torch.cuda.Event(enable_timing=True)
    events = []

    def step(record):
        e = [ev() for _ in range(4)]
        e[0].record()
        P.keygen(r_in, r_out, 0, rank * count, keys=(k0, k1))
        e[1].record()
        P.eval_fused_both(k0, k1, xhat, bits if sh["T"] else None, coeff if sh["has_lut"] else None)
        e[2].record()
        P.post_fused(k0, k1, xhat, bits[0], bits[1], coeff[0], coeff[1], outs=outs)
        e[3].record()
        if record:
            events.append(e)
    for _ in range(max(warmup, 3)):
        step(False)
    barrier()
    l0 = F.launch_count()
    start, stop = ev(), ev()
    start.record()
    for _ in range(steps):
        step(True)
    stop.record()
    barrier()
    ms = max_over_ranks(start.elapsed_time(stop)) / steps
    t_gen = sum(e[0].elapsed_time(e[1]) for e in events) / steps
    t_eval = sum(e[1].elapsed_time(e[2]) for e in events) / steps
    t_post = sum(e[2].elapsed_time(e[3]) for e in events) / steps
    aes_eval = cost["eval_cmp_aes"] + cost["eval_lut_aes"]
    lk_eval = cost["eval_cmp_lookups"] + cost["eval_lut_lookups"]
    ach = aes_eval * count / (t_eval / 2 * 1e-3) / 1e9
    peak = 148 * SM_CLOCK_MAX_MHZ * 1e6 * LDS_LANES_PER_CLK_SM / (lk_eval / max(1, aes_eval)) / 1e9
    key_b = P.key_bytes(1 << 20) / (1 << 20)
    return {"construction": ("variant 1 + bit 2: payload (1, -r, .., (-r)^d), coefficients of xhat^j, Horner in the public xhat: zero Beaver rounds (DESIGN 11)" if xpoly else
                             "variant 1: one DCF key f_{r,1} per view width, evaluated at the public points xhat + delta_j with shared tree prefixes (DESIGN 9)"),
            "post_rounds": P.post_rounds(),
            "value": world * count / (ms * 1e-3), "unit": "elements/s", "ms_per_step": ms,
            "eval_elems_per_s": world * count / (t_eval * 1e-3), "keygen_elems_per_s": world * count / (t_gen * 1e-3),
            "ms_breakdown": {"keygen": t_gen, "eval_fused_x2": t_eval, "post_fused": t_post},
            "key_bytes_per_elem_per_party": key_b, "online_bytes_per_elem_per_party": P.online_bits() / 8,
            "aes_per_elem": {"eval_one_party": aes_eval, "keygen_both": cost["gen_cmp_aes"] + cost["gen_lut_aes"]},
            "gpu_launches": F.launch_count() - l0,
            "projection": project((t_eval + t_post) / 2, P.online_bits() / 8 * count, 1 + P.post_rounds()),
            "roofline": {"bound": "alu", "kernel": "k_eval_sp", "achieved": ach, "peak": peak, "unit": "GAES/s (AES-128 blocks per second)",
                         "frac": ach / peak, "lookups_per_aes": lk_eval / max(1, aes_eval), "launch_ms": t_eval / 2,
                         "traffic": None if xpoly else NCU_TRAFFIC.get((name, count, "k_eval_sp")),
                         "hbm_achieved_gbs": key_b * count / (t_eval / 2 * 1e-3) / 1e9}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="gelu", help="config name in workloads.specs.CONFIGS (default: configs[1], GeLU 128x3072)")
    ap.add_argument("--count", type=int, default=0, help="override the element count (0 = the config's full tensor)")
    ap.add_argument("--chunk", type=int, default=0, help="elements per keygen/eval chunk (0 = whole tensor resident)")
    ap.add_argument("--ref-sample", type=int, default=512)
    ap.add_argument("--cpu-sample", type=int, default=4096)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sp", action="store_true", help="skip the variant-1 (shared-prefix) measurement")
    ap.add_argument("--blocks", action="store_true", help="also time the softmax vector block (config 3 shape: 12 x 128 rows of 128)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    if not os.path.exists(os.path.join(ROOT, "paper_2606_09551_b200", "libfusefss.so")):
        import __graft_entry__
        if local == 0:
            __graft_entry__.build()                                   # source-only checkout: compile the library first (no fallback)
        else:
            for _ in range(600):                                      # other ranks of this node wait for local rank 0's build
                if os.path.exists(os.path.join(ROOT, "paper_2606_09551_b200", "libfusefss.so")):
                    break
                time.sleep(1.0)
            time.sleep(2.0)
    import paper_2606_09551_b200 as F
    from workloads import specs, tensors

    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the product has no CPU fallback"
    torch.cuda.set_device(local)
    use_dist = world > 1 or "LOCAL_RANK" in os.environ          # under torchrun the group exists even for one rank
    if use_dist:
        if os.environ.get("NCCL_DEBUG", "VERSION").upper() == "VERSION":
            os.environ["NCCL_DEBUG"] = "WARN"                 # keep stdout to the one JSON line (no NCCL version banner)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    name = args.workload
    spec = specs.CONFIGS[name]()
    count = args.count or tensors.FULL_COUNT[name]
    P = F.Program(spec)
    sh = P.shape
    inp = tensors.inputs(name, spec, count=count, seed=rank)        # every rank: its own tensor of the config's shape
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    r_in, r_out, xhat = dev(inp["r_in"]), dev(inp["r_out"]), dev(inp["xhat"])
    chunk = args.chunk or count
    free_b, _ = torch.cuda.mem_get_info()
    while 2 * P.key_bytes(chunk) > 0.8 * free_b:                     # config 5 does not fit resident: stream in chunks
        chunk = (chunk + 1) // 2
    chunk = min(count, max(32, chunk))
    k0, k1 = P.alloc_keys(chunk)
    na = max(1, sh["n_out_a"])
    bits = [torch.empty(count, dtype=torch.int64, device="cuda") for _ in (0, 1)]
    coeff = [torch.empty((sh["p"], chunk), dtype=torch.int64, device="cuda") for _ in (0, 1)]
    youts = [torch.empty((na, chunk), dtype=torch.int64, device="cuda") for _ in range(2)]
    zouts = [torch.empty(chunk, dtype=torch.int64, device="cuda") for _ in range(2)]
    ev = lambda: torch.cuda.Event(enable_timing=True)
    t_gen, t_cmp, t_lut, t_post, t_genvec, t_genbit = [], [], [], [], [], []

    def step(record):
        for first in range(0, count, chunk):
            c = min(chunk, count - first)
            sl = slice(first, first + c)
            gfirst = rank * count + first                       # global element index: rank r owns [r*count, (r+1)*count)
            e = [ev() for _ in range(7)]
            ro = r_out[:, sl].contiguous() if spec.mask_output else r_out
            e[0].record()
            P.keygen(r_in[sl], ro, step.seed, gfirst, keys=(k0, k1), parts=1)          # T bit-DCF keys      (k_gen_bit)
            e[5].record()
            P.keygen(r_in[sl], ro, step.seed, gfirst, keys=(k0, k1), parts=2)          # M-1 vector-DCF keys (k_gen_vec)
            e[6].record()
            P.keygen(r_in[sl], ro, step.seed, gfirst, keys=(k0, k1), parts=4)          # share splitting     (k_gen_misc)
            e[1].record()
            if sh["T"]:
                for b, k in ((0, k0), (1, k1)):
                    P.eval_cmp(b, k, xhat[sl], out=bits[b][sl])
            e[2].record()
            cs = [None, None]
            if sh["has_lut"]:
                for b, k in ((0, k0), (1, k1)):
                    cs[b] = P.eval_lut(b, k, xhat[sl], out=coeff[b] if c == chunk else None)
            e[3].record()
            P.post_fused(k0, k1, xhat[sl], bits[0][sl], bits[1][sl], cs[0], cs[1],
                         outs=(youts[0], youts[1], zouts[0], zouts[1]) if c == chunk else None)
            e[4].record()
            if record:
                step.events.append(e)
    step.seed, step.events = 0, []

    def _allmax(v):
        if use_dist:
            t = torch.tensor([v], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return v

    def barrier():
        torch.cuda.synchronize()
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step(False)
    barrier()
    launches0 = F.launch_count()
    start, stop = ev(), ev()
    with ClockSampler(local) as clocks:
        start.record()
        for _ in range(args.steps):
            step(True)
        stop.record()
        barrier()
    launches = F.launch_count() - launches0
    ms = start.elapsed_time(stop)
    if use_dist:
        t = torch.tensor([ms], device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    for e in step.events:
        t_gen.append(e[0].elapsed_time(e[1])); t_cmp.append(e[1].elapsed_time(e[2]))
        t_lut.append(e[2].elapsed_time(e[3])); t_post.append(e[3].elapsed_time(e[4]))
        t_genbit.append(e[0].elapsed_time(e[5])); t_genvec.append(e[5].elapsed_time(e[6]))
    per_step = lambda ts: sum(ts) / args.steps
    ms_step = ms / args.steps
    value = world * count / (ms_step * 1e-3)

    # ---- roofline: AES-block rate of the dominant kernel against the shared-memory lookup roof (DESIGN 5.2) ----
    aes_eval, aes_gen = aes_per_elem(sh, spec.n)
    Q = (sh["p"] + 1) // 2
    n_chunks = len(step.events)
    full_chunk_frac = count / (chunk * ((count + chunk - 1) // chunk))      # tail chunk: fewer blocks per launch
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    key_b = P.key_bytes(1 << 20) / (1 << 20)
    lut_key_bytes = (8 * sh["p"] + (sh["M"] - 1) * (16 + spec.n * (16 + 8 * sh["p"]) + 8 * sh["p"])) if sh["has_lut"] else 0

    def grp(B):                                   # table lookups of B blocks that share their round-1 input (DESIGN 5.2)
        return 15 + B + 144 * B if B > 1 else 160

    def roof(kernel, aes_per_launch_elem, launches_per_chunk, times, bytes_per_elem, lookups_per_elem):
        lookups_per_aes = lookups_per_elem / max(1, aes_per_launch_elem)
        peak = 148 * SM_CLOCK_MAX_MHZ * 1e6 * LDS_LANES_PER_CLK_SM / lookups_per_aes / 1e9
        n_launch = launches_per_chunk * n_chunks
        launch_ms = sum(times) / max(1, n_launch)
        per_launch = aes_per_launch_elem * chunk * full_chunk_frac
        ach = per_launch / (launch_ms * 1e-3) / 1e9 if launch_ms > 0 else 0.0
        gbs = bytes_per_elem * chunk * full_chunk_frac / (launch_ms * 1e-3) / 1e9 if launch_ms > 0 else 0.0
        return {"bound": "alu", "kernel": kernel, "achieved": ach, "peak": peak,
                "unit": "GAES/s (AES-128 blocks per second)", "lookups_per_aes": lookups_per_aes,
                "frac": ach / peak, "traffic": NCU_TRAFFIC.get((name, count, kernel)),
                "peak_derivation": "148 SMs x 1.965 GHz x 32 conflict-free shared-memory lanes/clk/SM / lookups_per_aes (160 per block, less the round-1 lookups shared by blocks of one seed; DESIGN 5.2)",
                "launch_ms": launch_ms, "aes_per_launch": per_launch, "share_of_step": sum(times) / (ms_step * args.steps),
                "hbm_achieved_gbs": gbs, "hbm_peak_gbs": hbm_peak, "hbm_frac": gbs / hbm_peak,
                "hbm_peak_source": "measured (MEASURED_PEAKS.json)" if peaks else "fallback"}
    vec_gen_aes = (sh["M"] - 1) * (4 * spec.n * (1 + Q) + 2 * Q + 2) if sh["has_lut"] else 0
    vec_eval_aes = (sh["M"] - 1) * (spec.n * (1 + Q) + Q) if sh["has_lut"] else 0
    vec_gen_lookups = (sh["M"] - 1) * (2 * spec.n * grp(2 * (1 + Q)) + 2 * grp(Q) + 2 * 160) if sh["has_lut"] else 0
    vec_eval_lookups = (sh["M"] - 1) * (spec.n * grp(1 + Q) + grp(Q)) if sh["has_lut"] else 0
    roofs = {"k_gen_vec": roof("k_gen_vec", vec_gen_aes, 1, t_genvec, 2 * (lut_key_bytes - 8 * sh["p"]), vec_gen_lookups),
             "k_eval_lut": roof("k_eval_lut", vec_eval_aes, 2, t_lut, lut_key_bytes, vec_eval_lookups)}
    dominant = max(roofs.values(), key=lambda r: r["share_of_step"])
    roofline = dict(dominant)
    roofline["other_kernels"] = {k: {kk: v[kk] for kk in ("achieved", "frac", "launch_ms", "share_of_step", "hbm_achieved_gbs")}
                                 for k, v in roofs.items() if v is not dominant}
    for k, v in roofs.items():
        if v is not dominant:
            roofline["other_kernels"][k]["traffic"] = v["traffic"]

    line = {"metric": METRIC, "value": value, "unit": "elements/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64",
            "data": "synthetic",
            "config": {"workload": f"{name} n={spec.n} f={spec.f} count={count}", "chunk": chunk, "T": sh["T"], "M": sh["M"], "p": sh["p"],
                       "l2": "inputs_exceed_l2 (key material streamed once per step: %.1f GB per party)" % (P.key_bytes(chunk) / 1e9),
                       "parallelism": f"elements sharded over {world} GPU(s), no collective"},
            "eval_elems_per_s": world * count / ((per_step(t_cmp) + per_step(t_lut)) * 1e-3),
            "eval_post_elems_per_s": world * count / ((per_step(t_cmp) + per_step(t_lut) + per_step(t_post)) * 1e-3),
            "keygen_elems_per_s": world * count / (per_step(t_gen) * 1e-3),
            "ms_breakdown": {"keygen": per_step(t_gen), "keygen_bit": per_step(t_genbit), "keygen_vec": per_step(t_genvec), "eval_cmp_x2": per_step(t_cmp), "eval_lut_x2": per_step(t_lut), "post_fused": per_step(t_post)},
            "key_bytes_per_elem_per_party": key_b, "online_bytes_per_elem_per_party": P.online_bits() / 8,
            "online_bytes_per_elem_per_party_input_masked_mul": F.Program(specs.input_masked_mul(spec)).online_bits() / 8,
            "aes_per_elem": {"eval_one_party": aes_eval, "keygen_both": aes_gen},
            "aes_rate_gaes": {"eval": 2 * aes_eval * count / ((per_step(t_cmp) + per_step(t_lut)) * 1e-3) / 1e9,
                              "keygen": aes_gen * count / (per_step(t_gen) * 1e-3) / 1e9},
            "projection": project((per_step(t_cmp) + per_step(t_lut) + per_step(t_post)) / 2, P.online_bits() / 8 * count, 1 + P.post_rounds()),
            "gpu_launches": launches, "clocks": clocks.summary(), "roofline": roofline}

    # ---- PRG core alone (a pure AES chain, no key traffic): what the table design sustains on this GPU ----
    try:
        probe_threads, probe_iters = 148 * 1024 * 4, 192
        pout = torch.empty(probe_threads * 16, dtype=torch.uint8, device="cuda")
        F.aes_probe(probe_threads, probe_iters, pout)
        torch.cuda.synchronize()
        p0, p1 = ev(), ev()
        p0.record(); F.aes_probe(probe_threads, probe_iters, pout); p1.record()
        torch.cuda.synchronize()
        line["prg_probe"] = {"gaes": probe_threads * probe_iters / (p0.elapsed_time(p1) * 1e-3) / 1e9,
                             "what": "fusefss_aes_probe: 3 blocks per trip sharing round 1 (150 lookups per block), no key loads",
                             "lookup_roof_gaes": 148 * SM_CLOCK_MAX_MHZ * 1e6 * LDS_LANES_PER_CLK_SM / 150.0 / 1e9}
        del pout
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        pbuf = torch.empty(sms * 1024, dtype=torch.int32, device="cuda")
        for kind, key in ((0, "lop3_lane_ops_per_clk_per_sm"), (1, "lds32_lanes_per_clk_per_sm")):
            it = 4096
            F._check(F.lib.fusefss_pipe_probe(kind, it, pbuf.data_ptr(), torch.cuda.current_stream().cuda_stream))
            torch.cuda.synchronize()
            p0.record()
            F._check(F.lib.fusefss_pipe_probe(kind, it, pbuf.data_ptr(), torch.cuda.current_stream().cuda_stream))
            p1.record()
            torch.cuda.synchronize()
            line["prg_probe"][key] = sms * 1024 * 8 * it / (p0.elapsed_time(p1) * 1e-3) / (SM_CLOCK_MAX_MHZ * 1e6) / sms
        line["prg_probe"]["pipes"] = "fusefss_pipe_probe at 1.965 GHz: LOP3 chains (nominal 64 lanes/clk/SM) and conflict-free LDS.32 (nominal 32 lanes/clk/SM)"
    except Exception as exc:                                      # the probe is informative only
        line["prg_probe"] = {"error": str(exc)}

    # ---- the same workload with the single-key shared-prefix construction (variant 1) ------------------
    if not args.no_sp:
        del k0, k1, coeff, youts, zouts
        torch.cuda.empty_cache()
        line["shared_prefix"] = measure_shared_prefix(F, torch, name, spec, inp, rank, world, args.steps, args.warmup, barrier,
                                                      lambda v: (float(_allmax(v))))
        if spec.d >= 1:
            line["shared_prefix_public_horner"] = measure_shared_prefix(F, torch, name, spec, inp, rank, world, args.steps, args.warmup,
                                                                        barrier, lambda v: (float(_allmax(v))), xpoly=True)
        k0, k1 = None, None

    # ---- softmax vector block built from compiled gates (NEXT-3; DESIGN 12) ---------------------------------
    if args.blocks:
        from paper_2606_09551_b200 import blocks as gblocks
        rows, cols = 12 * 128, 128
        rngb = np.random.default_rng(5)
        xr = np.maximum(-20.0, -4.0 * rngb.exponential(1.0, size=(rows, cols))); xr[:, 0] = 0.0
        xq = np.floor(xr.reshape(-1) * 4096 + 0.5).astype(np.int64).view(np.uint64)
        U = lambda k: rngb.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rngb.integers(0, 2, size=k, dtype=np.uint64)
        x0h = U(xq.size)
        masks = {k: dev(U(c)) for k, c in (("nexp", xq.size), ("tr_e", xq.size), ("recip", rows), ("tr_t", rows), ("tr_y", xq.size))}
        blk = {}
        for v in (3, 0):
            B = gblocks.Softmax(rows, cols, v)
            x0d, x1d = dev(x0h), dev(xq - x0h)
            for _ in range(3):
                B.keygen(masks, 9); out = B.run(x0d, x1d)
            torch.cuda.synchronize()
            eb = [ev() for _ in range(3)]
            eb[0].record()
            for _ in range(args.steps):
                B.keygen(masks, 9)
            eb[1].record()
            for _ in range(args.steps):
                out = B.run(x0d, x1d)
            eb[2].record()
            torch.cuda.synchronize()
            y = (out["y"][0] + out["y"][1]).cpu().numpy().astype(np.float64).reshape(rows, cols) / 4096.0
            ref = np.exp(xr) / np.exp(xr).sum(axis=1, keepdims=True)
            blk["variant_%d" % v] = {"rows": rows, "cols": cols, "dealer_ms": eb[0].elapsed_time(eb[1]) / args.steps,
                                     "online_ms": eb[1].elapsed_time(eb[2]) / args.steps,
                                     "online_elems_per_s": rows * cols / (eb[1].elapsed_time(eb[2]) / args.steps * 1e-3),
                                     "key_bytes_per_elem_per_party": B.key_bytes_per_party() / (rows * cols),
                                     "online_bytes_per_elem_per_party": B.online_bytes_per_party() / (rows * cols), "rounds": B.rounds(),
                                     "max_abs_err_vs_float_softmax": float(np.abs(y - ref).max())}
            del B
            torch.cuda.empty_cache()
        line["softmax_block"] = blk
        rows, d = 1024, 1024                                              # config 4b's shape: 1024 tokens, d_model 1024
        xr = rngb.normal(0.0, 2.0, size=(rows, d))
        xq = np.floor(xr.reshape(-1) * 4096 + 0.5).astype(np.int64).view(np.uint64)
        x0h = U(xq.size)
        masks = {k: dev(U(c)) for k, c in (("mean", rows), ("var", rows), ("rsqrt", rows), ("tr_g", rows), ("tr_y", xq.size))}
        B = gblocks.LayerNorm(rows, d, 3)
        x0d, x1d = dev(x0h), dev(xq - x0h)
        for _ in range(3):
            B.keygen(masks, 9); out = B.run(x0d, x1d)
        torch.cuda.synchronize()
        eb = [ev() for _ in range(3)]
        eb[0].record()
        for _ in range(args.steps):
            B.keygen(masks, 9)
        eb[1].record()
        for _ in range(args.steps):
            out = B.run(x0d, x1d)
        eb[2].record()
        torch.cuda.synchronize()
        y = (out["y"][0] + out["y"][1]).cpu().numpy().astype(np.float64).reshape(rows, d) / 4096.0
        xf = xq.view(np.int64).astype(np.float64).reshape(rows, d) / 4096.0
        ref = (xf - xf.mean(axis=1, keepdims=True)) / xf.std(axis=1, keepdims=True)
        line["layernorm_block"] = {"variant_3": {"rows": rows, "d": d, "dealer_ms": eb[0].elapsed_time(eb[1]) / args.steps,
                                   "online_ms": eb[1].elapsed_time(eb[2]) / args.steps,
                                   "online_elems_per_s": rows * d / (eb[1].elapsed_time(eb[2]) / args.steps * 1e-3),
                                   "key_bytes_per_elem_per_party": B.key_bytes_per_party() / (rows * d),
                                   "online_bytes_per_elem_per_party": B.online_bytes_per_party() / (rows * d), "rounds": B.rounds(),
                                   "max_abs_err_vs_float_layernorm": float(np.abs(y - ref).max())}}
        del B
        torch.cuda.empty_cache()

    # ---- e2e: the public host-buffer call, pinned host memory, H2D + D2H inside the timed region -------
    if not args.no_e2e:
        e2e_chunk = min(chunk, 131072)
        ws = torch.empty(P.workspace_bytes(e2e_chunk), dtype=torch.uint8, device="cuda")
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).pin_memory()
        h_rin, h_rout, h_xhat = pin(inp["r_in"]), pin(inp["r_out"]), pin(inp["xhat"])
        hy = [torch.empty((na, count), dtype=torch.int64).pin_memory() for _ in range(2)]
        hz = [torch.zeros(count, dtype=torch.int64).pin_memory() for _ in range(2)]

        def e2e_step():
            F._check(F.lib.fusefss_gate_host(P._h, h_rin.data_ptr(), h_rout.data_ptr(), h_xhat.data_ptr(), 0, count, e2e_chunk,
                                             ws.data_ptr(), hy[0].data_ptr(), hy[1].data_ptr(), hz[0].data_ptr(), hz[1].data_ptr(),
                                             torch.cuda.current_stream().cuda_stream))
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            e2e_step()                                                  # synchronises its stream before returning
        barrier()
        dt = time.perf_counter() - t0
        if use_dist:
            t = torch.tensor([dt], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        h2d = count * 8 * (2 + (na if spec.mask_output else 0))
        d2h = count * 8 * (2 * sh["n_out_a"] + (2 if sh["n_out_b"] else 0))
        line["e2e"] = {"value": world * count * args.steps / dt, "unit": "elements/s", "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "api": "fusefss_gate_host (pinned host buffers, chunk=%d)" % e2e_chunk}
        # sanity: the e2e outputs reconstruct (first elements) -- not timed
        line["e2e"]["checksum_y"] = int((hy[0][0, :4] + hy[1][0, :4]).sum().item()) & 0xFFFFFFFF
        if not args.no_sp:                                              # the same public call on the variant-1 program
            Psp = F.Program(specs.shared_prefix(spec))
            sp_chunk = min(count, 1 << 20)
            ws2 = torch.empty(Psp.workspace_bytes(sp_chunk), dtype=torch.uint8, device="cuda")

            def e2e_sp():
                F._check(F.lib.fusefss_gate_host(Psp._h, h_rin.data_ptr(), h_rout.data_ptr(), h_xhat.data_ptr(), 0, count, sp_chunk,
                                                 ws2.data_ptr(), hy[0].data_ptr(), hy[1].data_ptr(), hz[0].data_ptr(), hz[1].data_ptr(),
                                                 torch.cuda.current_stream().cuda_stream))
            e2e_sp()
            barrier()
            t0 = time.perf_counter()
            for _ in range(args.steps):
                e2e_sp()
            barrier()
            dt2 = _allmax(time.perf_counter() - t0)
            line["shared_prefix"]["e2e"] = {"value": world * count * args.steps / dt2, "unit": "elements/s", "h2d_bytes_per_step": h2d,
                                            "d2h_bytes_per_step": d2h, "api": "fusefss_gate_host (pinned host buffers, chunk=%d)" % sp_chunk,
                                            "checksum_y": int((hy[0][0, :4] + hy[1][0, :4]).sum().item()) & 0xFFFFFFFF}
    if rank == 0 and not args.no_cpu and world >= 1:
        v, extra = cpu_oracle_rate(name, args.cpu_sample)
        line["cpu_baseline"] = {"value": v, "unit": "elements/s", "cores": 1, "kind": "oracle",
                                "sample": f"first {args.cpu_sample} elements of {name} (seed 0), whole gate: keygen + eval both parties + post; {extra['seconds']:.1f} s",
                                "keygen_elems_per_s": extra["keygen_elems_per_s"], "eval_post_elems_per_s": extra["eval_post_elems_per_s"]}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
