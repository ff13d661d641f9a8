#!/usr/bin/env python
"""bench.py -- one JSON line per run (driver contract + tier framing).

A "step" = one pass of the WHOLE hot path over the workload's tensor: fusefss_keygen (both key bundles; timed as its three
parts so that every kernel is bracketed by CUDA events), ONE fusefss_eval_fused_both call (packed comparison + interval lookup
for party 0 and party 1) and fusefss_post_fused.  The default workload is BASELINE.json configs[4] -- SiLU on Z_2^64, f = 12,
2048 x 11008 = 22,544,384 elements, the largest single-GPU configuration -- streamed in chunks whose two key buffers fit in
HBM (the Protocol-3 keys of the whole tensor are 3.3 TB).  `value` = elements/s of that whole step with the inputs resident in
HBM; eval-only and keygen-only rates, key and online bytes per element and the roofline of the dominant kernel ride along.
The same workload compiled with the single-key shared-prefix construction (`shared_prefix`, `shared_prefix_public_horner`),
the other six BASELINE tensors (`configs`), the PRG / pipe probes and the Eq. 1 LAN/WAN projection are measured in the same
run.  `e2e` = the same gate through fusefss_gate_host with pinned HOST buffers (H2D + D2H inside the timed region).
`--impl reference` times the CPU oracle instead.
N > 1 (torchrun): --scaling weak (default): every rank runs its own full tensor, value = N * count / max-over-ranks time;
--scaling strong: the tensor is sharded with paper_2606_09551_b200.sharding.shard_range.  No data-path collective either way
(elements are independent gate instances).
"""
from __future__ import annotations

import argparse
import gc
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
LDS_LANES_PER_CLK_SM = 32       # shared-memory crossbar: 128 B/clk/SM = 32 conflict-free 4-byte lanes (B300_MICROARCH "LDS/STS")
SMALL_COUNT = 1 << 16           # tensors up to this size: CUDA-graph replay per step + an L2 flush between timed steps


def project(t_comp_ms, bytes_per_party, rounds):
    """Eq. 1 of the paper: T_proj = T_comp + 2 B_comm / BW + R RTT, with its LAN / WAN parameters."""
    return {"t_comp_ms": t_comp_ms, "bytes_per_party": bytes_per_party, "rounds": rounds,
            "lan_ms": t_comp_ms + 2e3 * bytes_per_party / 1e9 + rounds * 0.5,
            "wan_ms": t_comp_ms + 2e3 * bytes_per_party / 400e6 + rounds * 4.0}


def load_json(path, default):
    try:
        with open(path) as f:
            return json.load(f)
    except Exception:
        return default


class Machine:
    """Roofline denominators: SM count from the device, SM clock and HBM bandwidth from MEASURED_PEAKS.json (driver-written),
    else the profiling guide's fallback; ncu DRAM traffic per launch from profiles/traffic.json."""

    def __init__(self, torch, local):
        self.peaks = load_json(os.path.join(ROOT, "MEASURED_PEAKS.json"), {})
        self.sms = torch.cuda.get_device_properties(local).multi_processor_count
        self.sm_mhz = float(self.peaks.get("sm_max_mhz") or 1965.0)
        self.hbm_gbs = float(self.peaks.get("hbm_gbs") or 6650.0)
        self.source = "measured (MEASURED_PEAKS.json)" if self.peaks else "fallback (B200_PROFILING.md: 1965 MHz, 6650 GB/s)"
        self.traffic = load_json(os.path.join(ROOT, "profiles", "traffic.json"), {})

    def lookup_peak_gaes(self, lookups_per_aes):
        return self.sms * self.sm_mhz * 1e6 * LDS_LANES_PER_CLK_SM / lookups_per_aes / 1e9

    def traffic_of(self, name, variant, count, kernel):
        return self.traffic.get(f"{name}/v{variant}/{count}/{kernel}")


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


# ---- the CPU oracle, as it stands, on the host cores ---------------------------------------------------------------------
def _oracle_chunk(args):
    """One chunk of the bounded sample: whole gate on the oracle (keygen + eval of both parties + post).  Runs in a thread: the
    oracle is single-threaded C behind ctypes, which releases the GIL."""
    O, inp, lo, hi, seed = args
    t0 = time.perf_counter()
    k0, k1 = O.keygen(inp["r_in"][lo:hi], np.ascontiguousarray(inp["r_out"][:, lo:hi]), seed, first_elem=lo)
    t1 = time.perf_counter()
    O.run_gate(k0, k1, inp["xhat"][lo:hi])
    return t1 - t0, time.perf_counter() - t1


def cpu_oracle_rate(name, sample, seed=0, threads=1):
    """Elements/s of the oracle on `sample` elements of workload `name`, on `threads` host threads (chunks of the sample run
    concurrently; each call is the unmodified single-threaded oracle)."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    from workloads import specs, tensors
    spec = specs.CONFIGS[name]()
    O = oracle.Program(spec)
    inp = tensors.inputs(name, spec, count=sample, seed=seed)
    threads = max(1, min(threads, sample))
    step = (sample + threads - 1) // threads
    jobs = [(O, inp, lo, min(sample, lo + step), seed) for lo in range(0, sample, step)]
    t0 = time.perf_counter()
    if threads == 1:
        parts = [_oracle_chunk(j) for j in jobs]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(_oracle_chunk, jobs))
    wall = time.perf_counter() - t0
    per = max(1, step)
    gen_s, ev_s = sum(p[0] for p in parts) / len(parts), sum(p[1] for p in parts) / len(parts)
    return sample / wall, dict(keygen_elems_per_s=per / gen_s if gen_s else None, eval_post_elems_per_s=per / ev_s if ev_s else None,
                               seconds=wall, threads=threads)


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the same workload (tier framing)."""
    if rank != 0:
        return
    sample = args.ref_sample
    cores = os.cpu_count() or 1
    vals = []
    for i in range(args.warmup + args.steps):
        v, _ = cpu_oracle_rate(args.workload, sample, seed=i, threads=cores)
        if i >= args.warmup:
            vals.append(sample / v)
    value = sample * len(vals) / sum(vals)
    from workloads import specs, tensors
    spec = specs.CONFIGS[args.workload]()
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "elements/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(vals) / len(vals),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": f"{args.workload} n={spec.n} f={spec.f} count={args.count or tensors.FULL_COUNT[args.workload]}",
                       "construction": "variant 0 (the paper's Protocol 3)", "sample": f"first {sample} elements per step"},
            "cpu_baseline": {"value": value, "unit": "elements/s", "cores": cores, "kind": "oracle",
                             "sample": f"{sample} elements of {args.workload} per step, whole gate (keygen + eval both parties + post), {cores} threads over elements"},
            "e2e": {"value": value, "unit": "elements/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---- one workload on the GPU ------------------------------------------------------------------------------------------------
class Gate:
    """A compiled gate type with its tensor on the device and every buffer a step needs (allocated once)."""

    def __init__(self, F, torch, name, variant, count, seed, first_global=0, chunk=0, spec_count=None):
        from workloads import specs, tensors
        self.F, self.torch, self.name, self.variant = F, torch, name, variant
        spec = specs.CONFIGS[name]()
        if variant & 1:
            spec = specs.shared_prefix(spec)
        if variant & 2:
            spec = specs.input_masked_mul(spec)
        if variant & 4:
            spec = specs.public_point_horner(spec)
        if variant & 8:
            spec = specs.early_termination(spec)
        if variant & 16:
            spec = specs.dense_table(spec)                               # lookup by full-domain evaluation (needs bit 0, n <= 16; DESIGN 14)
        self.spec, self.P = spec, F.Program(spec)
        self.sh, self.cost = self.P.shape, self.P.cost()
        self.count, self.first_global = count, first_global
        inp = tensors.inputs(name, spec, count=spec_count or count, seed=seed)
        if spec_count:                                                   # strong scaling: this rank's slice of the full tensor
            sl = slice(first_global, first_global + count)
            inp = {k: (v[..., sl] if k != "real" else v[sl]) for k, v in inp.items()}
        self.inp = inp
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
        self.r_in, self.r_out, self.xhat = dev(inp["r_in"]), dev(inp["r_out"]), dev(inp["xhat"])
        chunk = chunk or count
        gc.collect()
        torch.cuda.empty_cache()
        free_b, _ = torch.cuda.mem_get_info()
        per_elem = 8 * (6 + 2 * self.sh["p"] + 3 * max(1, self.sh["n_out_a"]))
        while 2 * self.P.key_bytes(chunk) + per_elem * chunk > 0.8 * free_b:     # does not fit resident: stream in chunks
            chunk = (chunk + 1) // 2
        if chunk < count:
            chunk = max(32, chunk // 32 * 32)
        self.chunk = chunk = min(count, chunk)
        self.k0, self.k1 = self.P.alloc_keys(chunk)
        na = max(1, self.sh["n_out_a"])
        I = lambda *shape: torch.empty(shape, dtype=torch.int64, device="cuda")
        self.bits = [I(chunk), I(chunk)]
        self.coeff = [I(self.sh["p"], chunk), I(self.sh["p"], chunk)]
        self.outs = (I(na, chunk), I(na, chunk), I(chunk), I(chunk))
        self.n_chunks = (count + chunk - 1) // chunk

    def free(self):
        for k in ("k0", "k1", "bits", "coeff", "outs", "r_in", "r_out", "xhat"):
            setattr(self, k, None)
        self.torch.cuda.empty_cache()

    def _views(self, first):
        c = min(self.chunk, self.count - first)
        sl = slice(first, first + c)
        ro = self.r_out[:, sl].contiguous() if self.spec.mask_output else self.r_out
        full = c == self.chunk
        bits = self.bits if full else [b[:c] for b in self.bits]
        coeff = self.coeff if full else [t.reshape(-1)[: self.sh["p"] * c].view(self.sh["p"], c) for t in self.coeff]
        outs = self.outs if full else None
        return c, sl, ro, bits, coeff, outs

    def keygen(self, first, parts):
        c, sl, ro, *_ = self._views(first)
        self.P.keygen(self.r_in[sl], ro, 0, self.first_global + first, keys=(self.k0, self.k1), parts=parts)

    def evaluate(self, first):
        c, sl, ro, bits, coeff, _ = self._views(first)
        if self.sh["T"] or self.sh["has_lut"]:
            self.P.eval_fused_both(self.k0, self.k1, self.xhat[sl], bits if self.sh["T"] else None, coeff if self.sh["has_lut"] else None)
        return bits, coeff

    def post(self, first, bits, coeff):
        c, sl, ro, _, _, outs = self._views(first)
        self.P.post_fused(self.k0, self.k1, self.xhat[sl], bits[0], bits[1], coeff[0], coeff[1], outs=outs)

    def step(self, events=None):
        ev = lambda: self.torch.cuda.Event(enable_timing=True)
        for first in range(0, self.count, self.chunk):
            e = [ev() for _ in range(6)] if events is not None else None
            rec = (lambda i: e[i].record()) if e else (lambda i: None)
            if e is None and self.count <= SMALL_COUNT:      # small tensors: the user's call, fusefss_keygen (tiny ones: ONE dealer launch)
                self.keygen(first, 7)
            else:
                rec(0); self.keygen(first, 1)            # the T bit-DCF keys (k_gen_bit)
                rec(1); self.keygen(first, 2)            # the lookup keys (k_gen_vec)
                rec(2); self.keygen(first, 4)            # share splitting (k_gen_misc)
            rec(3); bits, coeff = self.evaluate(first)
            rec(4); self.post(first, bits, coeff)
            rec(5)
            if e:
                events.append(e)


def _graph_of(torch, fn):
    """capture fn (library calls on torch's current stream) in a CUDA graph, after two eager warm-up calls on a side stream"""
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(2):
            fn()
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    return g


def _timed_graph(torch, g, flush, warmup, steps, median=False):
    """mean (or median) ms of `steps` replays, each bracketed by its own event pair with an L2 flush (a write larger than L2) before it"""
    for _ in range(warmup):
        g.replay()
    ts = []
    for _ in range(steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); g.replay(); b.record()
        ts.append((a, b))
    torch.cuda.synchronize()
    v = sorted(a.elapsed_time(b) for a, b in ts)
    return v[len(v) // 2] if median else sum(v) / steps


def small_sweep(F, torch):
    """--small-sweep: evaluation latency of BASELINE's small tensors against the forced number of warps an element's trees / points
    are dealt to (fusefss_debug_set force_g, sp_np) and the library's automatic choice; one JSON line per (tensor, construction).
    Evidence for the launch-geometry model in launch_eval_sp / pick_groups (profiles/r2e_small_sweep.md)."""
    from workloads import tensors
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for name in ("recip", "rsqrt", "relu16"):
        for variant in (1, 0):
            gate = Gate(F, torch, name, variant, tensors.FULL_COUNT[name], seed=0)
            gate.keygen(0, 7)
            run = lambda: _timed_graph(torch, _graph_of(torch, lambda: gate.evaluate(0)), flush, 3, 20, median=True)
            F.debug_set("force_g", 0); F.debug_set("sp_np", 0)
            line = {"name": name, "variant": variant, "count": gate.count, "auto_us": round(run() * 1e3, 1), "forced": {}}
            gmax = 20 if variant else max(gate.sh["M"] - 1, gate.sh["T"], 1)
            for g in range(1, gmax + 1):
                F.debug_set("force_g", g)
                for np_ in ((1, 2) if variant else (0,)):
                    F.debug_set("sp_np", np_)
                    line["forced"]["G%d_np%d" % (g, np_)] = round(run() * 1e3, 1)
            F.debug_set("force_g", 0); F.debug_set("sp_np", 0)
            print(json.dumps(line), flush=True)
            gate.free()


def measure(gate, M, steps, warmup, barrier, allmax, world=1, clocks_index=None):
    """Times `steps` steps of `gate`.  Large tensors: K steps inside one bracket (barrier + synchronize on both sides), per-kernel
    CUDA events inside.  Small tensors (<= SMALL_COUNT elements): the step is captured in a CUDA graph (launch-bound otherwise),
    each replay bracketed by its own event pair with an L2 flush in between; the phases are timed the same way from their own
    graphs."""
    torch, F, P, sh, cost = gate.torch, gate.F, gate.P, gate.sh, gate.cost
    count = gate.count
    ev = lambda: torch.cuda.Event(enable_timing=True)
    small = count <= SMALL_COUNT and gate.n_chunks == 1
    phases = {}
    clocks = None
    floor_ms = None
    if not small:
        for _ in range(warmup):
            gate.step()
        barrier()
        events = []
        start, stop = ev(), ev()
        sampler = ClockSampler(clocks_index) if clocks_index is not None else None
        if sampler:
            sampler.__enter__()
        l0 = F.launch_count()
        start.record()
        for _ in range(steps):
            gate.step(events)
        stop.record()
        barrier()
        if sampler:
            sampler.__exit__()
            clocks = sampler.summary()
        launches = F.launch_count() - l0
        ms_step = allmax(start.elapsed_time(stop)) / steps
        names = ("keygen_bit", "keygen_vec", "keygen_misc", "eval_both", "post_fused")
        for i, nm in enumerate(names):
            phases[nm] = sum(e[i].elapsed_time(e[i + 1]) for e in events) / steps
        l2 = "inputs_exceed_l2 (key material streamed once per step: %.1f GB per party per chunk)" % (P.key_bytes(gate.chunk) / 1e9)
    else:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

        graph_of = lambda fn: _graph_of(torch, fn)
        timed = lambda g: _timed_graph(torch, g, flush, warmup, steps)
        held = {}

        def ev_fn():
            held["bc"] = gate.evaluate(0)
        g_step = graph_of(lambda: gate.step())
        l_before = F.launch_count()
        gate.step()
        launches = (F.launch_count() - l_before) * steps
        barrier()
        sampler = ClockSampler(clocks_index) if clocks_index is not None else None
        if sampler:
            sampler.__enter__()
        ms_step = allmax(timed(g_step))
        if sampler:
            sampler.__exit__()
            clocks = sampler.summary()
        # the phases, each from its own graph, the same way (keys / inputs come from HBM after the flush)
        phases["keygen_bit"] = timed(graph_of(lambda: gate.keygen(0, 1))) if (sh["T"] and (not gate.variant & 1 or any(k < gate.spec.n for k in sh["k"]))) else 0.0
        phases["keygen_vec"] = timed(graph_of(lambda: gate.keygen(0, 2))) if sh["has_lut"] or gate.variant & 1 else 0.0
        phases["keygen_misc"] = timed(graph_of(lambda: gate.keygen(0, 4)))
        # the dealer call the STEP makes (fusefss_keygen, all parts): for tiny tensors that is ONE k_gen_tiny launch, a different kernel
        # from the three part launches above, which stay as a diagnostic (their sum exceeds this phase)
        l_gen = F.launch_count()
        gate.keygen(0, 7)
        dealer_launches = F.launch_count() - l_gen
        keygen_all_ms = timed(graph_of(lambda: gate.keygen(0, 7)))
        phases["eval_both"] = timed(graph_of(ev_fn))
        bits, coeff = held["bc"]
        phases["post_fused"] = timed(graph_of(lambda: gate.post(0, bits, coeff)))
        # latency floor of the evaluation: ONE 32-element tile per party through the same call (every tree / point group on its own
        # warp): the sequential chain of one element's walk + launch, table fill and the grid barrier.  A tensor this small cannot run
        # faster than that, whatever the machine's throughput (DESIGN 6 "small tensors").
        g1 = Gate(F, torch, gate.name, gate.variant, 32, seed=1)
        g1.keygen(0, 7)
        floor_ms = timed(graph_of(lambda: g1.evaluate(0)))
        g1.free()
        # Floors that do NOT come from the kernel under test (fusefss_aes_chain_probe: one warp, no key loads, no tree logic): every evaluation
        # of an element has to walk at least ONE root-to-leaf path of an n-level tree, level after level.  `independent`: a lane does all B blocks
        # of a level itself (the lane-per-element mapping: B = 1 + Q payload blocks per node); `strict`: one block per level on the lane's
        # dependent chain, the level's other blocks on other lanes (what any mapping short of splitting a single AES block across lanes can
        # reach).  Both include what every launch pays (launch + filling the 128-KB table window of a 256-thread CTA), timed the same way.
        if gate.variant & 1:
            pk = (cost["eval_lut_key_bytes"] - 16 - 16 * gate.spec.n) // (8 * gate.spec.n + 8) if cost["eval_lut_key_bytes"] else 1
        else:
            pk = sh["p"]
        level_blocks = min(5, 1 + (int(pk) + 1) // 2)
        pout = torch.empty(32 * 16, dtype=torch.uint8, device="cuda")
        indep_floor_ms = timed(graph_of(lambda: F.aes_chain_probe(level_blocks, gate.spec.n, pout)))
        strict_floor_ms = timed(graph_of(lambda: F.aes_chain_probe(1, gate.spec.n, pout)))
        launch_fill_ms = timed(graph_of(lambda: F.aes_chain_probe(1, 1, pout)))
        del flush
        l2 = "small tensor: CUDA-graph replay per step, a 256 MB L2 flush between timed replays (keys are read from HBM)"
    t_gen = phases["keygen_bit"] + phases["keygen_vec"] + phases["keygen_misc"]
    parts_note = None
    if small:                                                  # phases of the step as it runs: keygen_all + eval_both + post_fused
        parts_note = {"keygen_bit": phases.pop("keygen_bit"), "keygen_vec": phases.pop("keygen_vec"), "keygen_misc": phases.pop("keygen_misc"),
                      "what": "fusefss_keygen_parts launches timed alone (diagnostic: not the kernels the step runs when dealer_launches == 1)"}
        phases = {"keygen_all": keygen_all_ms, **phases}
        t_gen = keygen_all_ms
    t_eval, t_post = phases["eval_both"], phases["post_fused"]
    eval_aes = 2 * (cost["eval_cmp_aes"] + cost["eval_lut_aes"])
    eval_lk = 2 * (cost["eval_cmp_lookups"] + cost["eval_lut_lookups"])
    eval_key_bytes = 2 * (cost["eval_cmp_key_bytes"] + cost["eval_lut_key_bytes"])
    gen_aes = cost["gen_cmp_aes"] + cost["gen_lut_aes"]
    n_launch = gate.n_chunks
    per_launch_elems = count / n_launch
    eval_kernel = ("k_eval_dense" if gate.variant & 16 else "k_eval_sp") if gate.variant & 1 else "k_eval_p3"
    part_ms = parts_note or phases

    def roof(kernel, aes_elem, lk_elem, ms_total, bytes_elem):
        if not aes_elem or ms_total <= 0:
            return None
        launch_ms = ms_total / n_launch
        ach = aes_elem * per_launch_elems / (launch_ms * 1e-3) / 1e9
        peak = M.lookup_peak_gaes(lk_elem / aes_elem)
        gbs = bytes_elem * per_launch_elems / (launch_ms * 1e-3) / 1e9
        return {"bound": "alu", "pipe": "lsu_shared (the shared-memory data pipe: T-table lookups; ncu pipe_lsu 96.6 %, pipe_alu 81 % on k_gen_vec<3>)",
                "kernel": kernel, "achieved": ach, "peak": peak, "unit": "GAES/s (AES-128 blocks per second)",
                "frac": ach / peak, "lookups_per_aes": lk_elem / aes_elem, "launch_ms": launch_ms, "aes_per_launch": aes_elem * per_launch_elems,
                "share_of_step": ms_total / ms_step, "traffic": M.traffic_of(gate.name, gate.variant, int(per_launch_elems), kernel),
                "algorithmic_bytes_per_launch": bytes_elem * per_launch_elems,
                "hbm_achieved_gbs": gbs, "hbm_peak_gbs": M.hbm_gbs, "hbm_frac": gbs / M.hbm_gbs}
    roofs = {eval_kernel: roof(eval_kernel, eval_aes, eval_lk, t_eval, eval_key_bytes + 8 * (1 + 2 * (1 + sh["p"]))),
             "k_gen_vec": roof("k_gen_vec", cost["gen_lut_aes"], cost["gen_lut_lookups"], part_ms["keygen_vec"], 2 * cost["eval_lut_key_bytes"]),
             "k_gen_bit": roof("k_gen_bit", cost["gen_cmp_aes"], cost["gen_cmp_lookups"], part_ms["keygen_bit"], 2 * cost["eval_cmp_key_bytes"])}
    roofs = {k: v for k, v in roofs.items() if v}
    if small:                                                  # the whole dealer call against the roof of all its AES work; the part roofs are diagnostics
        for k in ("k_gen_vec", "k_gen_bit"):
            if k in roofs:
                roofs[k]["note"] = "part launch timed alone (k_gen_vec_quad / k_gen_bit): the step itself runs fusefss_keygen, see keygen_all"
        gen_lk = cost["gen_cmp_lookups"] + cost["gen_lut_lookups"]
        r_all = roof("k_gen_tiny" if dealer_launches == 1 else "fusefss_keygen (%d launches)" % dealer_launches, gen_aes, gen_lk, keygen_all_ms,
                     2 * (cost["eval_cmp_key_bytes"] + cost["eval_lut_key_bytes"]))
        if r_all:
            roofs["keygen_all"] = r_all
    key_b = P.key_bytes(1 << 20) / (1 << 20)
    res = {"count": count, "chunk": gate.chunk, "T": sh["T"], "M": sh["M"], "p": sh["p"], "rounds": P.post_rounds(),
           "value": world * count / (ms_step * 1e-3), "ms_per_step": ms_step,
           "eval_elems_per_s": world * count / (t_eval * 1e-3) if t_eval > 0 else None,
           "eval_post_elems_per_s": world * count / ((t_eval + t_post) * 1e-3),
           "keygen_elems_per_s": world * count / (t_gen * 1e-3),
           "ms_breakdown": phases, "key_bytes_per_elem_per_party": key_b, "online_bytes_per_elem_per_party": P.online_bits() / 8,
           "aes_per_elem": {"eval_one_party": eval_aes // 2, "keygen_both": gen_aes},
           "gpu_launches": launches, "l2": l2, "roofs": roofs, "eval_kernel": eval_kernel,
           "projection": project((t_eval + t_post) / 2, P.online_bits() / 8 * count, 1 + P.post_rounds())}
    if clocks is not None:
        res["clocks"] = clocks
    if floor_ms:
        res["eval_latency_floor_ms"] = floor_ms
        res["eval_independent_floor_ms"] = indep_floor_ms
        res["eval_strict_floor_ms"] = strict_floor_ms
        res["floor_level_blocks"] = level_blocks
        res["launch_and_table_fill_ms"] = launch_fill_ms
    if parts_note:
        res["keygen_parts_diagnostic_ms"] = parts_note
        res["dealer_launches_per_step"] = dealer_launches
    return res


def compact(res):
    """the per-config summary carried in `configs`"""
    ek = res["roofs"].get(res["eval_kernel"])
    dom = max(res["roofs"].values(), key=lambda r: r["share_of_step"]) if res["roofs"] else None
    return {"count": res["count"], "chunk": res["chunk"], "T": res["T"], "M": res["M"], "p": res["p"],
            "step_elems_per_s": res["value"], "eval_elems_per_s": res["eval_elems_per_s"], "keygen_elems_per_s": res["keygen_elems_per_s"],
            "ms_per_step": res["ms_per_step"], "ms_breakdown": res["ms_breakdown"],
            "key_bytes_per_elem_per_party": res["key_bytes_per_elem_per_party"],
            "online_bytes_per_elem_per_party": res["online_bytes_per_elem_per_party"], "post_rounds": res["rounds"],
            "eval_roof_frac": ek["frac"] if ek else None, "eval_kernel": res["eval_kernel"], "eval_launch_ms": ek["launch_ms"] if ek else None,
            "dominant_kernel": dom["kernel"] if dom else None, "dominant_roof_frac": dom["frac"] if dom else None,
            "traffic": ek["traffic"] if ek else None, "timing": "graph+flush" if res["l2"].startswith("small") else "events",
            "eval_latency_floor_ms": res.get("eval_latency_floor_ms"), "dealer_launches_per_step": res.get("dealer_launches_per_step"),
            "keygen_parts_diagnostic_ms": res.get("keygen_parts_diagnostic_ms"),
            "eval_floor_over_achieved": (res["eval_latency_floor_ms"] / ek["launch_ms"]) if (ek and res.get("eval_latency_floor_ms")) else None,
            # independent floor: one probe warp walking one n-level path (launch + table fill + n dependent 3-block trips), see measure()
            "eval_independent_floor_ms": res.get("eval_independent_floor_ms"), "launch_and_table_fill_ms": res.get("launch_and_table_fill_ms"),
            "eval_independent_floor_over_achieved": (res["eval_independent_floor_ms"] / ek["launch_ms"]) if (ek and res.get("eval_independent_floor_ms")) else None,
            "eval_strict_floor_ms": res.get("eval_strict_floor_ms"), "floor_level_blocks": res.get("floor_level_blocks"),
            "eval_strict_floor_over_achieved": (res["eval_strict_floor_ms"] / ek["launch_ms"]) if (ek and res.get("eval_strict_floor_ms")) else None}


def measure_a2b(F, torch, steps, count=1 << 20):
    """A gate whose Phi has interactive A2B nodes (workloads.specs.a2b_demo on Z_2^64: three extractions at bits 63, 12 and 1 plus a local
    one, DESIGN 15) on `count` uniform ring elements: dealer, both FSS calls, and the post-processing both ways -- one
    fused launch for both parties (k_post_fused<true>) against the per-round API (k_post_round<true>: one launch per party per round, each
    re-filling the 192-KB PRG table window because A2B rounds walk comparison keys)."""
    from workloads import specs, tensors
    spec = specs.a2b_demo(64, 12)
    P = F.Program(spec)
    rng = np.random.default_rng(0)
    x, r_in = tensors.uniform_ring(rng, count, 64), tensors.uniform_ring(rng, count, 64)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    d_rin, d_rout, d_xhat = dev(r_in), dev(tensors.uniform_ring(rng, count, 64).reshape(1, count)), dev(x + r_in)
    keys = P.alloc_keys(count)
    I = lambda *shape: torch.empty(shape, dtype=torch.int64, device="cuda")
    bits, coeff = [I(count), I(count)], [I(P.shape["p"], count), I(P.shape["p"], count)]
    outs = (I(1, count), I(1, count), I(count), I(count))
    R = P.post_rounds()
    msg = [torch.zeros(max(256, P.msg_total(count)), dtype=torch.uint8, device="cuda") for _ in (0, 1)]

    def per_round():
        for q in range(R + 1):
            for b in (0, 1):
                P.post(b, keys[b], d_xhat, bits[b], coeff[b], q, msg[1 - b], msg[b], y=outs[b], z=outs[2 + b])
    legs = {"keygen": lambda: P.keygen(d_rin, d_rout, 0, keys=keys), "eval_both": lambda: P.eval_fused_both(keys[0], keys[1], d_xhat, bits, coeff),
            "post_fused": lambda: P.post_fused(keys[0], keys[1], d_xhat, bits[0], bits[1], coeff[0], coeff[1], outs=outs), "post_per_round": per_round}
    ms, launches = {}, {}
    for nm, fn in legs.items():
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        l0 = F.launch_count()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(steps):
            fn()
        b.record()
        torch.cuda.synchronize()
        ms[nm], launches[nm] = a.elapsed_time(b) / steps, (F.launch_count() - l0) // steps
    step_ms = ms["keygen"] + ms["eval_both"] + ms["post_fused"]
    return {"spec": "a2b_demo(n=64, f=12): m=3, p=%d, T=%d, %d interactive A2B nodes, %d rounds" % (P.shape["p"], P.shape["T"], 3, R), "count": count,
            "ms": ms, "launches": launches, "step_elems_per_s": count / (step_ms * 1e-3),
            "post_fused_elems_per_s": count / (ms["post_fused"] * 1e-3), "post_per_round_elems_per_s": count / (ms["post_per_round"] * 1e-3),
            "key_bytes_per_elem_per_party": P.key_bytes(count) / count, "online_bytes_per_elem_per_party": P.online_bits() / 8,
            "timing": "CUDA events around %d calls after 2 warm-up calls; inputs (%.1f GB of keys per party) exceed L2" % (steps, P.key_bytes(count) / 1e9)}


def run_probes(F, torch, M, local):
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}
    try:
        probe_threads, probe_iters = M.sms * 1024 * 4, 192
        pout = torch.empty(probe_threads * 16, dtype=torch.uint8, device="cuda")
        F.aes_probe(probe_threads, probe_iters, pout)
        torch.cuda.synchronize()
        p0, p1 = ev(), ev()
        p0.record(); F.aes_probe(probe_threads, probe_iters, pout); p1.record()
        torch.cuda.synchronize()
        out = {"gaes": probe_threads * probe_iters / (p0.elapsed_time(p1) * 1e-3) / 1e9,
               "what": "fusefss_aes_probe: 3 blocks per trip sharing round 1 (150 lookups per block), no key loads",
               "lookup_roof_gaes": M.lookup_peak_gaes(150.0)}
        del pout
        pbuf = torch.empty(M.sms * 1024, dtype=torch.int32, device="cuda")
        st = torch.cuda.current_stream().cuda_stream
        for kind, key, per_thread in ((0, "lop3_lane_ops_per_clk_per_sm", 8), (1, "lds32_lanes_per_clk_per_sm", 8)):
            it = 4096
            F._check(F.lib.fusefss_pipe_probe(kind, it, pbuf.data_ptr(), st))
            torch.cuda.synchronize()
            p0.record(); F._check(F.lib.fusefss_pipe_probe(kind, it, pbuf.data_ptr(), st)); p1.record()
            torch.cuda.synchronize()
            out[key] = M.sms * 1024 * per_thread * it / (p0.elapsed_time(p1) * 1e-3) / (M.sm_mhz * 1e6) / M.sms
        out["pipes"] = "fusefss_pipe_probe at %.0f MHz: LOP3 chains (nominal 64 lanes/clk/SM) and conflict-free LDS.32 (nominal 32 lanes/clk/SM)" % M.sm_mhz
        if hasattr(F, "bitslice_probe"):
            out["bitsliced"] = F.bitslice_probe()
    except Exception as exc:                                      # the probes are informative only
        out["error"] = str(exc)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="silu", help="config name in workloads.specs.CONFIGS (default: configs[4], SiLU 2048x11008)")
    ap.add_argument("--variant", type=int, default=0, help="construction of the headline leg (0 = the paper's Protocol 3)")
    ap.add_argument("--count", type=int, default=0, help="override the element count (0 = the config's full tensor)")
    ap.add_argument("--chunk", type=int, default=0, help="elements per keygen/eval chunk (0 = as many as fit)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--ref-sample", type=int, default=0, help="--impl reference: elements per step (0 = sized for ~10 s per step)")
    ap.add_argument("--cpu-sample", type=int, default=0, help="cpu_baseline: elements (0 = sized for ~15 s)")
    ap.add_argument("--side-steps", type=int, default=3, help="steps of the secondary legs (other constructions, other configs, e2e)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sp", action="store_true", help="skip the variant-1 / variant-5 legs")
    ap.add_argument("--no-configs", action="store_true", help="skip the other BASELINE tensors")
    ap.add_argument("--no-probes", action="store_true")
    ap.add_argument("--blocks", action="store_true", help="also time the softmax / LayerNorm vector blocks")
    ap.add_argument("--small-sweep", action="store_true", help="sweep the launch geometry of the small tensors' evaluation call (tuning evidence) and exit")
    ap.add_argument("--two-party", action="store_true", help="N = 2: party b on GPU b, real exchange of the opening buffers (two_party.run_party)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="process-group backend for N > 1 (gloo: exchanges staged through pinned host memory)")
    ap.add_argument("--same-gpu", action="store_true", help="all ranks use cuda:0 (needs --backend gloo: NCCL refuses two ranks on one device).  A functional "
                    "stand-in for a multi-GPU node where only one GPU is at hand: it exercises the sharding / exchange code, its timings say nothing about NVLink")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)                               # timing rule: W >= 3
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    from workloads import specs, tensors
    if args.impl == "reference":
        if not args.ref_sample:
            args.ref_sample = {"silu": 1024, "gelu": 2048, "nexp": 2048, "shift_relu": 16384}.get(args.workload, tensors.FULL_COUNT[args.workload])
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    if not os.path.exists(os.path.join(ROOT, "paper_2606_09551_b200", "libfusefss.so")):
        import __graft_entry__
        if local == 0:
            __graft_entry__.build()                                   # source-only checkout: compile the library first (no fallback)
        else:
            for _ in range(900):                                      # other ranks of this node wait for local rank 0's build
                if os.path.exists(os.path.join(ROOT, "paper_2606_09551_b200", "libfusefss.so")):
                    break
                time.sleep(1.0)
            time.sleep(2.0)
    import paper_2606_09551_b200 as F

    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the product has no CPU fallback"
    if args.same_gpu:
        assert args.backend == "gloo", "--same-gpu needs --backend gloo (NCCL refuses two ranks on one device)"
        local = 0
    torch.cuda.set_device(local)
    use_dist = world > 1 or "LOCAL_RANK" in os.environ          # under torchrun the group exists even for one rank
    red_dev = "cuda" if args.backend == "nccl" else "cpu"       # where the few scalars that cross ranks live
    if use_dist:
        if args.backend == "nccl":
            if os.environ.get("NCCL_DEBUG", "VERSION").upper() == "VERSION":
                os.environ["NCCL_DEBUG"] = "WARN"             # keep stdout to the one JSON line (no NCCL version banner)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")

    def allmax(v):
        if use_dist:
            t = torch.tensor([v], device=red_dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return v

    def allsum32(v):
        """sum over ranks of 32-bit checksums, mod 2^32"""
        if use_dist:
            t = torch.tensor([int(v)], device=red_dev, dtype=torch.int64)
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
            return int(t.item()) & 0xFFFFFFFF
        return int(v) & 0xFFFFFFFF

    def checksum_of(g):
        """32-bit checksum of the reconstructed outputs the gate's LAST chunk left on the device: sum_e (y0 + y1 mod 2^n) mod 2^32.  Randomness is
        indexed by the global element, so a tensor sharded over ranks (one chunk per rank) sums to the one-rank value."""
        c = g.count - (g.n_chunks - 1) * g.chunk
        y = g.outs[0][0, :c] + g.outs[1][0, :c]                 # int64 arithmetic wraps mod 2^64
        if g.spec.n < 64:
            y = y & ((1 << g.spec.n) - 1)
        return int((y & 0xFFFFFFFF).sum().item()) & 0xFFFFFFFF

    def barrier():
        torch.cuda.synchronize()
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    M = Machine(torch, local)
    if args.small_sweep:
        small_sweep(F, torch)
        return
    if args.two_party:
        from paper_2606_09551_b200 import two_party
        line = two_party.bench(F, torch, dist, args, rank, world, M)
        if rank == 0:
            print(json.dumps(line), flush=True)
        if use_dist:
            dist.barrier()
            dist.destroy_process_group()
        return

    name = args.workload
    full = args.count or tensors.FULL_COUNT[name]
    strong = args.scaling == "strong" and world > 1
    if strong:                                                      # the config's tensor sharded by contiguous element ranges
        from paper_2606_09551_b200 import sharding
        first, count = sharding.shard_range(full, rank, world)
        gate = Gate(F, torch, name, args.variant, count, seed=0, first_global=first, chunk=args.chunk, spec_count=full)
        eff_world, parallelism = 1, f"strong: {full} elements sharded over {world} GPU(s) by sharding.shard_range, no collective"
    else:                                                           # weak: every rank its own tensor of the config's shape
        count = full
        gate = Gate(F, torch, name, args.variant, count, seed=rank, first_global=rank * count, chunk=args.chunk)
        eff_world, parallelism = world, (f"replicas: each of {world} GPU(s) runs its own {count}-element tensor, no collective" if world > 1 else "1 GPU")
    res = measure(gate, M, args.steps, args.warmup, barrier, allmax, world=eff_world, clocks_index=local)
    if strong:
        res["value"] = full / (res["ms_per_step"] * 1e-3)
    out_sum = allsum32(checksum_of(gate)) if (strong or world == 1) else checksum_of(gate)
    spec, sh, P = gate.spec, gate.sh, gate.P
    dominant = max(res["roofs"].values(), key=lambda r: r["share_of_step"])
    roofline = dict(dominant)
    roofline["peak_derivation"] = ("%d SMs x %.0f MHz x 32 conflict-free shared-memory lanes/clk/SM / lookups_per_aes (160 per block, less the round-1 "
                                   "lookups shared by blocks of one seed; DESIGN 5.2); SM count from the device, clock from %s" % (M.sms, M.sm_mhz, M.source))
    roofline["other_kernels"] = {k: {kk: v[kk] for kk in ("achieved", "frac", "launch_ms", "share_of_step", "hbm_achieved_gbs", "traffic")}
                                 for k, v in res["roofs"].items() if v is not dominant}
    line = {"metric": METRIC, "value": res["value"], "unit": "elements/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "u64",
            "data": "synthetic",
            "config": {"workload": f"{name} n={spec.n} f={spec.f} count={full}",
                       "construction": f"variant {args.variant}" + (" (the paper's Protocol 3)" if args.variant == 0 else ""),
                       "chunk": gate.chunk, "chunks_per_step": gate.n_chunks, "T": sh["T"], "M": sh["M"], "p": sh["p"], "l2": res["l2"],
                       "parallelism": parallelism},
            "eval_elems_per_s": res["eval_elems_per_s"], "eval_post_elems_per_s": res["eval_post_elems_per_s"],
            "keygen_elems_per_s": res["keygen_elems_per_s"], "ms_breakdown": res["ms_breakdown"],
            "key_bytes_per_elem_per_party": res["key_bytes_per_elem_per_party"],
            "online_bytes_per_elem_per_party": res["online_bytes_per_elem_per_party"],
            "online_bytes_per_elem_per_party_input_masked_mul": F.Program(specs.input_masked_mul(spec)).online_bits() / 8,
            "aes_per_elem": res["aes_per_elem"], "projection": res["projection"], "gpu_launches": res["gpu_launches"],
            "clocks": res.get("clocks"), "roofline": roofline,
            "output_checksum": {"value": out_sum, "what": "sum over elements of (y0 + y1 mod 2^n) mod 2^32 of the last chunk" +
                                (", summed over the ranks' shards" if strong else (" (rank 0's replica)" if world > 1 else ""))}}
    if use_dist:
        line["config"]["backend"] = args.backend + (", all ranks on cuda:0 (functional stand-in, not an NVLink measurement)" if args.same_gpu else "")
    side_steps = max(1, min(args.steps, args.side_steps))
    inp_host = gate.inp

    # ---- e2e: the public host-buffer call, pinned host memory, H2D + D2H inside the timed region -------
    def e2e_of(prog, shp, chunk, steps):
        na = max(1, shp["n_out_a"])
        ws = torch.empty(prog.workspace_bytes(chunk), dtype=torch.uint8, device="cuda")
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).pin_memory()
        h_rin, h_rout, h_xhat = pin(inp_host["r_in"]), pin(inp_host["r_out"]), pin(inp_host["xhat"])
        hy = [torch.empty((na, count), dtype=torch.int64).pin_memory() for _ in range(2)]
        hz = [torch.zeros(count, dtype=torch.int64).pin_memory() for _ in range(2)]

        def one():
            F._check(F.lib.fusefss_gate_host(prog._h, h_rin.data_ptr(), h_rout.data_ptr(), h_xhat.data_ptr(), 0, count, chunk,
                                             ws.data_ptr(), ws.numel(), hy[0].data_ptr(), hy[1].data_ptr(), hz[0].data_ptr(), hz[1].data_ptr(),
                                             torch.cuda.current_stream().cuda_stream))
        one()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            one()                                                   # synchronises its stream before returning
        barrier()
        dt = allmax(time.perf_counter() - t0)
        h2d = count * 8 * (2 + (na if spec.mask_output else 0))
        d2h = count * 8 * (2 * shp["n_out_a"] + (2 if shp["n_out_b"] else 0))
        out = {"value": eff_world * count * steps / dt, "unit": "elements/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": steps, "api": "fusefss_gate_host (pinned host buffers, chunk=%d)" % chunk,
               "checksum_y": int((hy[0][0, :4] + hy[1][0, :4]).sum().item()) & 0xFFFFFFFF}
        del ws, one                                                 # the workspace (up to 103 GB) must be gone before the next leg sizes its buffers
        gc.collect()
        torch.cuda.empty_cache()
        return out
    gate_chunk, gate_chunks, gate_first = gate.chunk, gate.n_chunks, gate.first_global
    gate.free()                                                     # the e2e workspace holds its own key buffers
    if not args.no_e2e:
        e2e_chunk = gate_chunk if gate_chunks > 1 else min(count, 1 << 17)
        line["e2e"] = e2e_of(P, sh, e2e_chunk, max(3, side_steps) if res["ms_per_step"] > 2000 else side_steps)   # one untimed call, then >= 3 timed

    # ---- N > 1, replicas: the ONE tensor of the config sharded over the ranks as well, so that a scaling record carries a strong-scaling point
    if world > 1 and not strong:
        from paper_2606_09551_b200 import sharding
        f2, c2 = sharding.shard_range(full, rank, world)
        gs = Gate(F, torch, name, args.variant, c2, seed=0, first_global=f2, chunk=args.chunk, spec_count=full)
        rs = measure(gs, M, side_steps, 3, barrier, allmax, world=1)
        line["strong_scaling_leg"] = {"value": full / (rs["ms_per_step"] * 1e-3), "unit": "elements/s", "ms_per_step": rs["ms_per_step"], "steps": side_steps,
                                      "what": f"the config's one {full}-element tensor sharded over {world} ranks by sharding.shard_range (contiguous, 32-aligned ranges; "
                                              "randomness indexed by the global element; no collective); max-over-ranks time",
                                      "output_checksum": allsum32(checksum_of(gs)) if gs.n_chunks == 1 else None}
        gs.free()

    if not args.no_probes:
        line["prg_probe"] = run_probes(F, torch, M, local)
        lds = line["prg_probe"].get("lds32_lanes_per_clk_per_sm")
        if lds:                                                     # `frac` uses the nominal 32 lanes/clk/SM; this one the rate the pipe probe reached in this run
            line["roofline"]["frac_vs_measured_lds"] = line["roofline"]["frac"] * LDS_LANES_PER_CLK_SM / lds
            line["roofline"]["measured_lds_lanes_per_clk_per_sm"] = lds

    # ---- the same workload with the single-key shared-prefix construction (variants 1 and 5) ------------------
    if not args.no_sp and not (args.variant & 1):
        for key, v in (("shared_prefix", args.variant | 1), ("shared_prefix_public_horner", args.variant | 5)):
            if v & 4 and spec.d < 1:
                continue
            g2 = Gate(F, torch, name, v, count, seed=0 if strong else rank, first_global=gate_first, spec_count=full if strong else None)
            r2 = measure(g2, M, side_steps, 3, barrier, allmax, world=eff_world)
            ek = r2["roofs"][r2["eval_kernel"]]
            obj = {"construction": ("variant 5: variant 1 + payload (1, -r, .., (-r)^d), Horner in the public xhat: zero Beaver rounds (DESIGN 11)" if v & 4 else
                                    "variant 1: one DCF key f_{r,1} per view width, evaluated at the public points xhat + delta_j with shared tree prefixes (DESIGN 9)"),
                   "steps": side_steps}
            obj.update({k: r2[k] for k in ("value", "ms_per_step", "eval_elems_per_s", "keygen_elems_per_s", "ms_breakdown", "key_bytes_per_elem_per_party",
                                           "online_bytes_per_elem_per_party", "aes_per_elem", "gpu_launches", "projection", "chunk")})
            obj["unit"], obj["post_rounds"], obj["roofline"] = "elements/s", r2["rounds"], ek
            p2, s2 = g2.P, g2.sh
            g2.free()
            if key == "shared_prefix" and not args.no_e2e:
                obj["e2e"] = e2e_of(p2, s2, min(count, 1 << 20), side_steps)
            line[key] = obj

    # ---- the other BASELINE tensors (configs[0..3]), each at its full size, Protocol 3 and single-key -----------
    if not args.no_configs:
        cfgs = {}
        for other in specs.CONFIGS:
            if other == name:
                continue
            row = {}
            # variants 8 / 9 = 0 / 1 with early-terminated bit trees (DESIGN 13), on the tensors whose gates have comparison atoms worth cutting;
            # variant 17 = single key + dense-table lookup (DESIGN 14), on config 1 at its full 4,096 elements (n = 16)
            extra = (8, 9) if other in ("relu16", "shift_relu", "gelu") else ()
            extra += (17,) if other == "relu16" else ()
            for v in (0, 1) + extra:
                g3 = Gate(F, torch, other, v, tensors.FULL_COUNT[other], seed=0)
                row["variant_%d" % v] = compact(measure(g3, M, side_steps, 3, barrier, allmax))
                g3.free()
            cfgs[other] = row
        cfgs[name] = {"variant_%d" % args.variant: compact(res)}
        line["configs"] = cfgs
        line["a2b_gate"] = measure_a2b(F, torch, side_steps)

    if args.blocks:
        from paper_2606_09551_b200 import blocks as gblocks
        line.update(gblocks.bench(F, torch, side_steps))

    if rank == 0 and not args.no_cpu:
        cores = os.cpu_count() or 1
        v1, ex1 = cpu_oracle_rate(name, min(count, 128), threads=1)               # calibration: one thread, a few elements
        sample = args.cpu_sample or int(min(count, max(256, v1 * cores * 12.0)))    # ~12-15 s of work on all cores
        vN, exN = cpu_oracle_rate(name, sample, threads=cores)
        line["cpu_baseline"] = {"value": vN, "unit": "elements/s", "cores": cores, "kind": "oracle",
                                "sample": f"first {sample} elements of {name} (seed 0), whole gate: keygen + eval both parties + post; {exN['seconds']:.1f} s on {cores} threads over elements (the oracle itself is single-threaded C)",
                                "single_thread_elems_per_s": v1, "keygen_elems_per_s_per_thread": ex1["keygen_elems_per_s"],
                                "eval_post_elems_per_s_per_thread": ex1["eval_post_elems_per_s"]}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
