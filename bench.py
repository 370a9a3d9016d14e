#!/usr/bin/env python
"""bench.py — throughput of the WarpGuard check path on B200, one JSON line (contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 4] [--events E]

Workload (N = 1): BASELINE.json config 4, the mixed paper-shaped stream — 51,621 sites, 58.0 M warp events of
which 52.2 M are checks on protected sites (38.3 M return + 13.9 M forward), 0.05 % violations,
enforce mode — generated on the GPU by `streams.py` (seeded, synthetic; stands in for the paper's corpus).
A STEP is one pass of the whole hot path over that stream:
    wg_sign_continuations   (a1 a2 a3 a7)      backward push of every return event
    wg_verify_continuations (a1 a2 a4-a8)      check_ret + forward membership + verdicts + counters
`value` = checks on protected sites per second over the whole step (sign time included), inputs resident in HBM.
`e2e` = the same step through the *_host C-ABI calls: events in pinned HOST memory, H2D / D2H inside the timed
region, on a bounded prefix of the same stream.  `cpu_baseline` = the oracle, as it stands, single-threaded, on a
bounded prefix of the same stream (and its verdicts are compared with the GPU's while we are at it).

Under torchrun (N > 1) ONE config-4 stream is sharded: rank r checks the contiguous slice shard_range(n, r, N) with
its own engine (policy and key replicated, sequence base = slice start); no data-path collective — the only exchange is
the counter all-reduce at read-out, outside the hot loop; timing is max over ranks; "scaling": "strong".  `--weak` gives
every rank its own full stream instead ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "cfi_checks_per_sec"
UNIT = "checks/s"
# algorithmic integer work: 32-bit integer lane-operations
OPS_PER_MAC_VERIFY = 310   # 12 SipRounds x 24 + 13 injection + 7 finalisation + 2 compare
OPS_PER_MAC_SIGN = 308
# bytes per event
B_RET_VERIFY, B_RET_SIGN, B_FWD, B_NON = 536, 528, 280, 24
# DRAM traffic of the dominant kernel: read from the committed ncu --set full capture under profiles/ — never typed in
TRAFFIC_FILE = ROOT / "profiles" / "r02_traffic.json"
KERNEL_SOURCES = ["paper_2606_11871_b200/csrc/wg_check.cu", "paper_2606_11871_b200/csrc/wg_internal.h",
                  "include/warpguard_sip32.cuh"]


def kernel_source_hash() -> str:
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        h.update((ROOT / f).read_bytes())
    return h.hexdigest()[:16]


def measured_traffic(config: int, n_events: int):
    """(bytes per launch, source note) of the verify kernel from profiles/r02_traffic.json, or (None, why): the capture
    must be of THIS kernel source (hash) on this workload."""
    if not TRAFFIC_FILE.exists():
        return None, "no capture committed"
    try:
        t = json.loads(TRAFFIC_FILE.read_text())
    except Exception:
        return None, "profiles/r02_traffic.json unreadable"
    if t.get("source_hash") != kernel_source_hash():
        return None, "stale: kernel sources changed since the capture (%s, commit %s)" % (TRAFFIC_FILE.name, t.get("commit"))
    if t.get("config") != config or t.get("events") != n_events:
        return None, "capture is of config %s / %s events" % (t.get("config"), t.get("events"))
    return int(t["dram_bytes_read"]) + int(t["dram_bytes_write"]), "%s: ncu --set full at commit %s" % (TRAFFIC_FILE.name, t.get("commit"))


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--events", type=int, default=None, help="events per rank (default: the config's full size)")
    ap.add_argument("--e2e-events", type=int, default=8_000_000)
    ap.add_argument("--cpu-events", type=int, default=4_000_000)
    ap.add_argument("--ref-events", type=int, default=1_000_000, help="events per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--profile", type=int, default=0,
                    help="wg_set_profile flags for the timed calls (1 backward-only, 2 forward-only, 4 low-telemetry, "
                         "8 metadata integrity); the headline run uses 0")
    ap.add_argument("--batches", type=int, default=0,
                    help="config 5 only: stream that many 8 M-event batches (BASELINE.json: 64 = 512 M events), "
                         "alternating detect / enforce, and report the summed kernel time")
    ap.add_argument("--weak", action="store_true", help="N > 1: every rank checks its own full stream (weak scaling) "
                    "instead of a slice of one stream")
    ap.add_argument("--host-batches", type=int, default=4,
                    help="config 5 stream: batches also pushed through the *_host calls (wall time including H2D / D2H)")
    ap.add_argument("--source-hash", action="store_true", help="print the kernel source hash profiles/r02_traffic.json must carry")
    ap.add_argument("--shadow", action="store_true",
                    help="also time the stateful shadow stack (SURVEY 8(f-1)): one lock-step push + check_ret over 1 Mi warps")
    return ap.parse_args()


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text())
        except Exception:
            pass
    return {}


def probe_int_pipe(device: int, mix: int) -> float:
    """int32 lane-ops per second of the register-only integer probe (csrc/wg_probe.cu -> libwg_probe.so, a
    measurement helper that is not part of libwarpguard.so)."""
    import ctypes as C
    lib = C.CDLL(str(ROOT / "paper_2606_11871_b200" / "libwg_probe.so"))
    lib.wg_probe_int_pipe.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    ops, ms = C.c_double(0), C.c_double(0)
    err = lib.wg_probe_int_pipe(int(device), int(mix), C.byref(ops), C.byref(ms))
    if err != 0:
        raise RuntimeError(f"wg_probe_int_pipe: cudaError {err}")
    return ops.value


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("timestamp,uuid,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, uuid: str | None):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.uuid = (uuid or "").lower()
        cmd = ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"]
        try:
            self.p = subprocess.Popen(cmd, stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def window(self, t0, t1) -> None:
        """Only samples stamped inside [t0, t1] (datetime, local time) are kept: the timed region."""
        self.t0, self.t1 = t0, t1

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [[x.strip() for x in line.split(",")] for line in self.f.read().splitlines()]
        rows = [c for c in rows if len(c) >= 9]
        t0, t1 = getattr(self, "t0", None), getattr(self, "t1", None)
        if t0 is not None:
            import datetime as _dt
            kept = []
            for c in rows:
                try:
                    ts = _dt.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f")
                except ValueError:
                    continue
                if t0 <= ts <= t1:
                    kept.append(c)
            rows = kept or rows  # (a region shorter than one sampling period keeps the whole run's samples)
        rows = [c[1:] for c in rows]
        mine = [c for c in rows if self.uuid and self.uuid in c[0].lower()]
        for c in (mine or rows):  # this rank's GPU; every visible GPU if the uuid could not be matched
            c = c[1:]
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def forward_search_ops(st, torch, lo=0, hi=None) -> int:
    """(7 ceil(log2(n+1)) + 3) int32 ops per unique active target of every non-empty forward event
    (SURVEY.md §8(d)); unique targets = 1 for a warp-uniform event, min(popc(active), n) otherwise."""
    import numpy as np
    from paper_2606_11871_b200 import streams as S
    dev = st.hdr.device
    kind = torch.from_numpy(st.policy.kind.astype(np.int64)).to(dev)
    cnt = torch.from_numpy(np.diff(st.policy.tgt_off.astype(np.int64))).to(dev)
    site = st.site_id()[lo:hi]
    sel = kind[site] == S.PROTECTED_FORWARD
    n = cnt[site[sel]].double()
    mask = st.active_mask()[lo:hi][sel]
    pc = torch.zeros_like(mask)
    for b in range(32):
        pc += (mask >> b) & 1
    uniq = torch.where(st.uniform[lo:hi][sel], torch.ones_like(pc), torch.minimum(pc, n.long()))
    uniq = torch.where(pc > 0, uniq, torch.zeros_like(uniq))
    per = 7 * torch.ceil(torch.log2(n + 1)) + 3
    return int((per * uniq.double()).sum().item())


# ---------------------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------------
def run_reference(a) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return  # rank 0 alone runs and prints it
    import numpy as np
    import oracle
    from paper_2606_11871_b200 import streams as S

    st = S.make_stream(a.config, "cpu", n_events=a.ref_events)
    pol = st.policy
    orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, pol.policy_digest)
    hdr = st.hdr.numpy().view(np.uint64)
    tag_t = __import__("torch").from_numpy(orc.sign(hdr, st.val.numpy().view(np.uint64)).view(np.int64))
    st.apply_return_tamper(tag_t)
    val, tag = st.val.numpy().view(np.uint64), tag_t.numpy().view(np.uint64)

    def step():
        orc.sign(hdr, val)
        orc.verify(hdr, val, tag, st.mode)

    for _ in range(a.warmup):
        step()
    orc.reset_counters()
    t0 = time.perf_counter()
    for _ in range(a.steps):
        step()
    dt = time.perf_counter() - t0
    g, _ = orc.read_counters()
    checks = (g["ret_checks"] + g["fwd_checks"]) / a.steps
    lanes = (g["ret_lanes"] + g["fwd_lanes"]) / a.steps
    v = checks / (dt / a.steps)
    sample = f"{a.ref_events} events of config {a.config} per step (same recipe and proportions, seed of the config)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": 1e3 * dt / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "lane_verdicts_per_sec": lanes / (dt / a.steps),
        "config": {"workload": f"config{a.config}-{S.NAMES[a.config]}", "events_per_step": a.ref_events,
                   "step": "oracle sign + oracle verify", "note": "CPU oracle (g++ -O2, 1 thread); bounded sample"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------
def run_ours(a) -> None:
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2606_11871_b200 import binding as B
    from paper_2606_11871_b200 import sharding
    from paper_2606_11871_b200 import streams as S

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the check path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs, resident in HBM before anything is timed ----
    n_stream = S.FULL_EVENTS[a.config] if a.events is None else a.events
    if a.config == 5 and a.events is None:
        n_stream = S.CONFIG5_BATCH
    sharded = world > 1 and not a.weak
    # sharded (default for N > 1): every rank builds the SAME seeded stream and keeps its contiguous slice; weak: a
    # stream of its own per rank
    st = S.make_stream(a.config, dev, n_events=n_stream, batch_index=0 if sharded else rank)
    lo, hi = sharding.shard_range(n_stream, rank, world) if sharded else (0, n_stream)
    n_events = hi - lo
    eng = B.Engine(local).load(st.policy)
    tag_full = eng.wg_sign_continuations(st.hdr, st.val)     # tokens at push time (engine's own signer)
    st.apply_return_tamper(tag_full)                          # then the recorded corruption
    hdr, val, tag = st.hdr[lo:hi], st.val[lo:hi], tag_full[lo:hi]
    in_slice = lambda plan: int(((plan.ev >= lo) & (plan.ev < hi)).sum().item()) if len(plan) else 0  # noqa: E731
    planned_ret, planned_fwd = in_slice(st.ret_tamper), in_slice(st.fwd_tamper)
    if a.profile:
        eng.wg_set_profile(a.profile)
    tag_scratch = torch.empty_like(tag)
    out = torch.empty((n_events, 2), dtype=torch.int32, device=dev)
    fwd_ops = forward_search_ops(st, torch, lo, hi)
    # inputs smaller than the 126 MB L2 (config 1) would be re-read from L2 by every step: a 256 MB buffer is written
    # between the timed steps then; every other config streams far more than the L2 holds per step
    step_bytes = n_events * (B_RET_VERIFY + B_RET_SIGN)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if step_bytes < (512 << 20) else None
    torch.cuda.synchronize()

    def step():
        eng.wg_sign_continuations(hdr, val, tag_scratch)
        eng.wg_verify_continuations(hdr, val, tag, st.mode, out)

    # integer-pipe ceilings of this GPU, measured now (register-only probe)
    probes = {}
    for name, mix in (("iadd3", 0), ("lop3", 1), ("shf", 2), ("imad", 3), ("imad_wide", 4),
                      ("lop3+imad_1:1", 5), ("sipround_alu_mix", 6), ("imad_hi", 7), ("alu+imad_2:1", 8),
                      ("shf+imad_hi_1:1", 9), ("add64_pairs", 10), ("sipround_x24", 11)):
        probes[name] = probe_int_pipe(local, mix)

    props = torch.cuda.get_device_properties(local)
    uuid = str(props.uuid) if hasattr(props, "uuid") else None
    sampler = ClockSampler(uuid)  # started before the warm-up so that it is sampling when the timed region begins
    # W warm-up steps; the LAST of them is enqueued after the opening barrier, right in front of the timed steps, so
    # that the GPU is busy (clocks up, nothing idle) when the first timed step starts — the counters therefore cover
    # K + 1 identical steps
    for _ in range(max(a.warmup - 1, 0)):
        step()
    eng.wg_reset_counters()
    if sharded:
        eng.wg_set_sequence_base(lo)  # (a reset restarts the sequence; the slice keeps the stream's numbering)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(a.steps)]
    barrier()
    import datetime as _dt
    t_region0 = _dt.datetime.now()
    step()
    launches0 = eng.wg_kernel_launches()
    for k in range(a.steps):
        if flush is not None:
            flush.zero_()  # L2 flush, outside the event brackets
        ev[k][0].record()
        eng.wg_sign_continuations(hdr, val, tag_scratch)
        ev[k][1].record()
        eng.wg_verify_continuations(hdr, val, tag, st.mode, out)
        ev[k][2].record()
    barrier()
    sampler.window(t_region0, _dt.datetime.now())
    clocks = sampler.stop()
    launches = eng.wg_kernel_launches() - launches0
    step_list = [e[0].elapsed_time(e[2]) for e in ev]       # device time of each step (CUDA events on the launch stream)
    sign_list = [e[0].elapsed_time(e[1]) for e in ev]
    verify_list = [e[1].elapsed_time(e[2]) for e in ev]
    total_ms = sum(step_list)
    sign_ms = sum(sign_list) / a.steps
    verify_ms = sum(verify_list) / a.steps
    med = lambda x: sorted(x)[len(x) // 2]  # noqa: E731
    g, _ = eng.wg_read_counters(per_site=False)

    # ---- what one step judged (counters accumulated over K identical steps) ----
    K = a.steps
    KC = K + 1  # steps the counters saw (the last warm-up step runs after the reset)
    for k in ("ret_checks", "fwd_checks", "ret_lanes", "fwd_lanes", "ret_viol_events", "fwd_viol_events"):
        assert g[k] % KC == 0, (k, g[k])
    checks = (g["ret_checks"] + g["fwd_checks"]) // KC
    lanes = (g["ret_lanes"] + g["fwd_lanes"]) // KC
    # properties that hold at any size: every planned corruption is found, nothing else is
    if not (a.profile & 2):
        assert g["ret_viol_events"] // KC == planned_ret, (g["ret_viol_events"], planned_ret)
    if not (a.profile & 1):
        assert g["fwd_viol_events"] // KC == planned_fwd, (g["fwd_viol_events"], planned_fwd)
    assert g["events_total"] // KC == n_events
    ret_ev, fwd_ev = g["ret_checks"] // KC, g["fwd_checks"] // KC
    non_ev = n_events - ret_ev - fwd_ev

    t = torch.tensor([total_ms, sign_ms, verify_ms, med(step_list), min(step_list), med(verify_list), min(verify_list)],
                     dtype=torch.float64, device=dev)
    tot = torch.tensor([checks, lanes], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    total_ms, sign_ms, verify_ms, step_med, step_best, verify_med, verify_best = t.tolist()
    all_checks, all_lanes = tot.tolist()
    ms_per_step = total_ms / K
    value = all_checks / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (the check kernel of wg_verify_continuations) ----
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = props.multi_processor_count
    # one warp instruction per cycle per SM sub-partition = 128 int32 lane-ops / SM / clk when the
    # ALU pipe (64 / SM / clk) and the FMA pipe's IMAD (64 / SM / clk) are both fed; the larger of that derived
    # figure and every measured probe is the denominator, so a weak probe cannot flatter the fraction.
    derived_peak = 128.0 * n_sm * sm_max_mhz * 1e6
    # the SipRound probe is not a pipe peak but the ceiling of this instruction mix (20 of its 24 operations can
    # only issue on the ALU pipe at 2 cycles per warp instruction): reported beside the peak, never as the peak
    sip_ceiling = probes.get("sipround_x24", 0.0)
    alu_peak = max([derived_peak] + [v for k, v in probes.items() if k != "sipround_x24"])
    verify_ops = OPS_PER_MAC_VERIFY * (g["ret_lanes"] // KC) + fwd_ops
    verify_bytes = B_RET_VERIFY * ret_ev + B_FWD * fwd_ev + B_NON * non_ev
    sign_ops = OPS_PER_MAC_SIGN * (g["ret_lanes"] // KC)
    t_alu = verify_ops / alu_peak
    t_hbm = verify_bytes / (hbm_peak * 1e9)
    achieved = verify_ops / (verify_ms * 1e-3)
    traffic, traffic_src = measured_traffic(a.config, n_events) if world == 1 else (None, "one GPU only")
    roofline = {
        "kernel": "wg_check_kernel<verify> (wg_verify_continuations)",
        "bound": "alu" if t_alu >= t_hbm else "hbm",
        **({"achieved": achieved / 1e12, "peak": alu_peak / 1e12, "unit": "Tint32op/s", "frac": achieved / alu_peak}
           if t_alu >= t_hbm else
           {"achieved": verify_bytes / (verify_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
            "frac": verify_bytes / (verify_ms * 1e-3) / 1e9 / hbm_peak}),
        "alu_achieved_Tops": achieved / 1e12, "alu_frac": achieved / alu_peak,
        "traffic": traffic, "traffic_source": traffic_src,
        "ms_per_launch_median": verify_med, "ms_per_launch_best": verify_best,
        "ms_per_launch_steps": [round(x, 4) for x in verify_list],
        "peak_source": ("derived: 128 lanes/SM/clk x %d SMs x %.0f MHz (DESIGN.md §6); max with the measured probes"
                        % (n_sm, sm_max_mhz)),
        "ms_per_launch": verify_ms, "algorithmic_ops_per_launch": verify_ops,
        "algorithmic_bytes_per_launch": verify_bytes,
        "hbm_achieved_gbs": verify_bytes / (verify_ms * 1e-3) / 1e9, "hbm_peak_gbs": hbm_peak,
        "hbm_frac": verify_bytes / (verify_ms * 1e-3) / 1e9 / hbm_peak,
        "hbm_peak_source": "measured (MEASURED_PEAKS.json)" if "hbm_gbs" in peaks else "fallback",
        "t_roof_ms": 1e3 * max(t_alu, t_hbm), "frac_of_roof_time": max(t_alu, t_hbm) / (verify_ms * 1e-3),
        "sign_kernel": {"ms_per_launch": sign_ms, "achieved": sign_ops / (sign_ms * 1e-3) / 1e12,
                        "frac": sign_ops / (sign_ms * 1e-3) / alu_peak,
                        "hbm_achieved_gbs": (B_RET_SIGN * ret_ev + 16 * (n_events - ret_ev) + 256 * (n_events - ret_ev))
                        / (sign_ms * 1e-3) / 1e9},
        "sipround_ceiling": sip_ceiling / 1e12,
        "frac_of_sipround_ceiling": (achieved / sip_ceiling) if sip_ceiling else None,
        "note": ("achieved counts ALGORITHMIC int32 ops (310 per verified lane: 12 SipRounds); the kernel executes "
                 "fewer (site word and warp-uniform continuation word absorbed once per event, no round on an inactive "
                 "lane), so the fraction of the SipRound ceiling can exceed 1"),
        "probes_Tops": {k: v / 1e12 for k, v in probes.items()},
    }

    # ---- end to end: HOST buffers through the *_host C-ABI calls, copies inside the timed region ----
    e2e = None
    ne = min(a.e2e_events, n_events)
    h = {}
    if not a.no_e2e or not a.no_cpu_baseline:
        h["hdr"] = hdr[:ne].cpu().pin_memory()
        h["val"] = val[:ne].cpu().pin_memory()
        h["tag"] = tag[:ne].cpu().pin_memory()
    if not a.no_e2e:
        h_scratch = torch.empty((ne, 32), dtype=torch.int64).pin_memory()
        h_out = torch.empty((ne, 2), dtype=torch.int32).pin_memory()

        def e2e_step():
            eng.wg_sign_continuations_host(h["hdr"], h["val"], h_scratch)
            eng.wg_verify_continuations_host(h["hdr"], h["val"], h["tag"], st.mode, h_out)

        torch.cuda.synchronize()  # (the *_host calls are not ordered after work pending on this stream)
        e2e_step()
        eng.wg_reset_counters()
        barrier()
        reps = 3
        t0 = time.perf_counter()
        for _ in range(reps):
            e2e_step()
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / reps
        ge, _ = eng.wg_read_counters(per_site=False)
        e_checks = (ge["ret_checks"] + ge["fwd_checks"]) / reps
        assert torch.equal(h_out, out[:ne].cpu()), "host-buffer path and device-buffer path disagree"
        te = torch.tensor([dt], dtype=torch.float64, device=dev)
        ce = torch.tensor([e_checks], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
            dist.all_reduce(ce, op=dist.ReduceOp.SUM)
        e2e = {"value": ce.item() / te.item(), "unit": UNIT,
               "h2d_bytes_per_step": ne * ((16 + 256) + (16 + 256 + 256)), "d2h_bytes_per_step": ne * (256 + 8),
               "events_per_step": ne, "ms_per_step": 1e3 * te.item(),
               "api": "wg_sign_continuations_host + wg_verify_continuations_host (pinned host buffers)"}

    # ---- the oracle beside it (rank 0, N = 1 only) ----
    cpu = None
    if not a.no_cpu_baseline and world == 1:
        import oracle
        nc = min(a.cpu_events, ne)
        pol = st.policy
        orc = oracle.Oracle(pol.kind, pol.tgt_off, pol.tgts, pol.k0, pol.k1, pol.policy_digest)
        hh, hv, ht = (h[k][:nc].numpy().view(np.uint64) for k in ("hdr", "val", "tag"))
        t0 = time.perf_counter()
        orc.sign(hh, hv)
        o_out = orc.verify(hh, hv, ht, st.mode)
        dt = time.perf_counter() - t0
        og, _ = orc.read_counters(per_site=False)
        same = np.array_equal(o_out, out[:nc].cpu().numpy().view(np.uint32))
        assert same, "GPU verdicts differ from the oracle on the cpu_baseline sample"
        cpu = {"value": (og["ret_checks"] + og["fwd_checks"]) / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"first {nc} events of the same stream, oracle sign + verify, {dt:.1f} s; "
                         f"verdicts equal the GPU's on all {nc} events",
               "lane_verdicts_per_sec": (og["ret_lanes"] + og["fwd_lanes"]) / dt}

    # ---- optional: the stateful shadow stack (wg_shadow_push + wg_shadow_check_ret), one lock-step call each ----
    shadow = None
    if a.shadow:
        ns, depth = 1 << 20, 4
        eng.wg_shadow_configure(ns, depth)
        gsh = torch.Generator(device=dev).manual_seed(4242)
        ret_sites = torch.from_numpy(np.nonzero(st.policy.kind == S.PROTECTED_RETURN)[0]).to(dev)
        site = ret_sites[torch.randint(0, len(ret_sites), (ns,), generator=gsh, device=dev)]
        slot = torch.randperm(ns, generator=gsh, device=dev)
        mask = st.active_mask()[:ns]
        s_hdr = torch.stack([site | (mask << 32), (1 << 48) | (slot << 5)], dim=1).contiguous()
        s_val = st.val[:ns].contiguous()
        s_out = torch.empty((ns, 2), dtype=torch.int32, device=dev)
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        for rep_ in range(4):  # each repetition pushes one frame and pops it again: the state returns to empty
            evs[0].record()
            eng.wg_shadow_push(s_hdr, s_val, st.mode, s_out)
            evs[1].record()
            eng.wg_shadow_check_ret(s_hdr, s_val, st.mode, s_out)
            evs[2].record()
        torch.cuda.synchronize()
        csh = eng.wg_shadow_read_counters()
        assert csh["viol_lanes"] == 0 and csh["push_lanes"] == csh["check_lanes"]
        lanes = csh["push_lanes"] // 4
        push_ms, chk_ms = evs[0].elapsed_time(evs[1]), evs[1].elapsed_time(evs[2])
        # bytes: header 16 + value row 256 + verdict 8 + per active lane: depth counter 4 r + 4 w, entry sector 32 (w or r)
        byts = ns * 280 + lanes * 40
        shadow = {"warps_per_call": ns, "max_depth": depth, "lanes_per_call": int(lanes),
                  "push_ms": push_ms, "check_ret_ms": chk_ms, "launches_per_call": 2,
                  "push_lanes_per_sec": lanes / (push_ms * 1e-3), "check_lanes_per_sec": lanes / (chk_ms * 1e-3),
                  "push_alu_frac": OPS_PER_MAC_SIGN * lanes / (push_ms * 1e-3) / alu_peak,
                  "check_alu_frac": OPS_PER_MAC_VERIFY * lanes / (chk_ms * 1e-3) / alu_peak,
                  "push_gbs": byts / (push_ms * 1e-3) / 1e9, "check_gbs": byts / (chk_ms * 1e-3) / 1e9}

    # ---- read-out exchange (outside the hot loop): counters summed over ranks ----
    gr, _ = sharding.reduce_counters(g, None, 0, device=dev)
    small = flush is not None
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": a.warmup,
            "ms_per_step": ms_per_step, "ms_per_step_median": step_med, "ms_per_step_best": step_best,
            "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "u64", "data": "synthetic",
            "lane_verdicts_per_sec": all_lanes / (ms_per_step * 1e-3),
            "verify_only_checks_per_sec": all_checks / (verify_ms * 1e-3),
            "config": {"workload": f"config{a.config}-{S.NAMES[a.config]}", "events_per_gpu": n_events, "events_total": n_stream if sharded else n_events * world,
                       "checks_per_step": int(all_checks), "lane_verdicts_per_step": int(all_lanes),
                       "n_sites": st.policy.n_sites, "mode": "enforce" if st.mode else "detect", "profile_flags": a.profile,
                       "step": "wg_sign_continuations + wg_verify_continuations over the whole stream",
                       "l2": ("a 256 MB buffer is written between the timed steps (the step's inputs, %.0f MB, would fit the "
                              "126 MB L2)" % ((verify_bytes + B_RET_SIGN * ret_ev) / 1e6)) if small else
                             ("inputs (%.1f GB per step per GPU) are far larger than the 126 MB L2; no flush needed"
                              % ((verify_bytes + B_RET_SIGN * ret_ev) / 1e9)),
                       "parallelism": "1 GPU" if world == 1 else
                       (f"{world} ranks, one stream of {n_stream} events sharded in contiguous slices, counters all-reduced "
                        "at read-out" if sharded else f"{world} ranks x own stream, counters all-reduced at read-out")},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
            **({"shadow": shadow} if shadow else {}),
            "counters": {k: gr[k] for k in ("events_total", "ret_checks", "fwd_checks", "ret_viol", "fwd_viol",
                                           "blocked_lanes", "first_violation_key")},
        }))
    eng.close()
    if world > 1:
        dist.destroy_process_group()


def run_config5_stream(a) -> None:
    """BASELINE.json config 5 as a stream: `--batches` batches of 8 M events over the 1 M-site policy (sets up to 4,096
    entries), detect on even and enforce on odd batches, each batch generated on the GPU, signed, corrupted and
    verified; kernel time summed over the batches (generation excluded).  A parity-test case measured, not the
    headline line: prints one JSON object."""
    import torch

    from paper_2606_11871_b200 import binding as B
    from paper_2606_11871_b200 import streams as S

    dev = torch.device("cuda", 0)
    pol = S.make_policy(5, dev)
    eng = B.Engine(0).load(pol)
    sign_ms = verify_ms = 0.0
    planned_ret = planned_fwd = events = 0
    out = tag = None
    for b in range(-1, a.batches):  # batch -1 is the warm-up
        st = S.make_stream(5, dev, policy=pol, batch_index=max(b, 0))
        n = st.hdr.shape[0]
        if out is None:
            out = torch.empty((n, 2), dtype=torch.int32, device=dev)
            tag = torch.empty((n, 32), dtype=torch.int64, device=dev)
        e0, e1, e2, e3 = (torch.cuda.Event(enable_timing=True) for _ in range(4))
        e0.record()
        eng.wg_sign_continuations(st.hdr, st.val, tag)
        e1.record()
        st.apply_return_tamper(tag)
        e2.record()
        eng.wg_verify_continuations(st.hdr, st.val, tag, st.mode, out)
        e3.record()
        torch.cuda.synchronize()
        if b < 0:
            eng.wg_reset_counters()
            continue
        sign_ms += e0.elapsed_time(e1)
        verify_ms += e2.elapsed_time(e3)
        planned_ret += len(st.ret_tamper)
        planned_fwd += len(st.fwd_tamper)
        events += n
        del st
    g, _ = eng.wg_read_counters(per_site=False)
    assert g["events_total"] == events and g["ret_viol_events"] == planned_ret
    assert planned_fwd - 20 * a.batches <= g["fwd_viol_events"] <= planned_fwd
    checks, lanes = g["ret_checks"] + g["fwd_checks"], g["ret_lanes"] + g["fwd_lanes"]

    # ---- the same stream from HOST memory: wall time including transfers (SURVEY 8(d) "Config 5 ... wall time including
    #      transfers, double-buffered on two streams"): a few batches pushed through the *_host calls, which stage 256 Ki
    #      event chunks alternately on two streams (H2D, kernels and D2H of consecutive chunks overlap) ----
    host = None
    if a.host_batches > 0:
        hb = min(a.host_batches, a.batches)
        wall = 0.0
        h_checks = 0
        h2d = d2h = 0
        for b in range(hb):
            st = S.make_stream(5, dev, policy=pol, batch_index=b)
            n = st.hdr.shape[0]
            eng.wg_sign_continuations(st.hdr, st.val, tag)
            st.apply_return_tamper(tag)
            torch.cuda.synchronize()
            h_hdr, h_val, h_tag = st.hdr.cpu().pin_memory(), st.val.cpu().pin_memory(), tag.cpu().pin_memory()
            h_scratch = torch.empty((n, 32), dtype=torch.int64).pin_memory()
            h_out = torch.empty((n, 2), dtype=torch.int32).pin_memory()
            eng.wg_reset_counters()
            t0 = time.perf_counter()
            eng.wg_sign_continuations_host(h_hdr, h_val, h_scratch)
            eng.wg_verify_continuations_host(h_hdr, h_val, h_tag, st.mode, h_out)
            wall += time.perf_counter() - t0
            gh, _ = eng.wg_read_counters(per_site=False)
            h_checks += gh["ret_checks"] + gh["fwd_checks"]
            assert gh["ret_viol_events"] == len(st.ret_tamper)
            h2d += n * ((16 + 256) + (16 + 256 + 256))
            d2h += n * (256 + 8)
            del st, h_hdr, h_val, h_tag, h_scratch, h_out
        host = {"batches": hb, "wall_ms_total": 1e3 * wall, "checks_per_sec": h_checks / wall,
                "h2d_bytes": h2d, "d2h_bytes": d2h, "gbytes_per_sec_both_ways": (h2d + d2h) / wall / 1e9,
                "api": "wg_sign_continuations_host + wg_verify_continuations_host (pinned host buffers)"}
    print(json.dumps({
        "workload": "config5-stress stream", "batches": a.batches, "events": events, "checks": checks,
        "lane_verdicts": lanes, "sign_ms_total": sign_ms, "verify_ms_total": verify_ms,
        "checks_per_sec_verify": checks / (verify_ms * 1e-3), "lane_verdicts_per_sec_verify": lanes / (verify_ms * 1e-3),
        "checks_per_sec_sign_plus_verify": checks / ((sign_ms + verify_ms) * 1e-3),
        "violations_found": {"ret_events": g["ret_viol_events"], "fwd_events": g["fwd_viol_events"],
                             "planned_ret": planned_ret, "planned_fwd": planned_fwd},
        "blocked_lanes": g["blocked_lanes"], "n_sites": pol.n_sites,
        "n_targets": int(pol.tgt_off[-1]), "host_stream": host}))
    eng.close()


def main():
    a = parse_args()
    if a.source_hash:
        print(kernel_source_hash())
        return
    if a.impl == "reference":
        run_reference(a)
    elif a.config == 5 and a.batches > 0:
        run_config5_stream(a)
    else:
        run_ours(a)


if __name__ == "__main__":
    main()
