#!/usr/bin/env python
"""bench.py -- whole verify-and-switch rounds of the WhiFlash hot path on synthetic data (B200).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--sub-workloads cfg2,cfg3,cfg4] [--impl reference]

A step is one round of the whole path over one batch: target-page
reserve, 36 layers of verify attention, accept/entropy/route, then the switch (wf_switch_round: eager
append for the active drafter, lazy enqueue for the idle one, flush for sequences the router switches,
all derived on the device from the route).  The headline workload is cfg5 (BASELINE.json configs[4],
the largest single-GPU config); cfg2-cfg4 ride on the same line as compact `per_config` sub-records.
One JSON line is printed by rank 0.  Multi-GPU: the path does not shard (BASELINE.json north_star: one GPU, no
collectives) -> "replicas only": every rank runs the same workload independently, timed as the max
over ranks.  `--impl reference` times the CPU oracle (oracle/) on a bounded sample instead.
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
sys.path.insert(0, ROOT)

from paper_2606_07710_b200 import synth  # noqa: E402

WORKLOADS = {"cfg1": 0, "cfg2": 1, "cfg3": 2, "cfg4": 3, "cfg5": 4}
# dram__bytes_read.sum + dram__bytes_write.sum per attention launch, from the committed `ncu --set full` capture named
# beside each figure (a profiler cannot run inside the timed region); workloads without a capture report null
NCU_TRAFFIC = {   # dram__bytes_read.sum + dram__bytes_write.sum per attention launch, from the committed ncu --set full captures
    "cfg5": (1059.9e6, "profiles/r2_final.md section 5 (ncu --set full of this workload, stream-K over 148 SMs, final round-2 library)"),
    "cfg2": (17.14e6, "profiles/r2_final.md section 5 (ncu --set full of this workload, 8 clusters of 10, final round-2 library)"),
    "cfg3": (548.2e6, "profiles/r2_final.md section 5 (ncu --set full of this workload, one CTA per pair, final round-2 library)"),
    "cfg4": (545.9e6, "profiles/r2_final.md section 5 (ncu --set full of this workload, 32 clusters of 4, final round-2 library)"),
}
METRIC = "verify_rounds_per_s"
UNIT = "rounds/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: NVML (what nvidia-smi reads) polled every 5 ms
    from a thread started before the warm-up; `nvidia-smi -lms` as the fallback.  mark() brackets the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None
        self.t_mark = []                  # host times bracketing the timed region (after a device sync each)
        self.stop_flag = False
        self.source = None

    def _phys_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            ids = [v.strip() for v in vis.split(",") if v.strip()]
            if self.index < len(ids) and ids[self.index].isdigit():
                return int(ids[self.index])
        return self.index

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self._phys_index())
            mx = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            bits = [pynvml.nvmlClocksThrottleReasonHwSlowdown, pynvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                    pynvml.nvmlClocksThrottleReasonSwThermalSlowdown, pynvml.nvmlClocksThrottleReasonSwPowerCap]

            def poll():
                while not self.stop_flag:
                    try:
                        sm = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                        r = int(pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                        self.rows.append((time.time(), sm, mx, [bool(r & b) for b in bits]))
                    except Exception:
                        pass
                    time.sleep(0.005)
            self.source = "nvml"
            self.thread = threading.Thread(target=poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            pass
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self._phys_index()), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.source = "nvidia-smi -lms 20"
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            if len(r) >= 6 and r[0].replace(".", "").isdigit():
                mx = float(r[1]) if r[1].replace(".", "").isdigit() else None
                self.rows.append((time.time(), float(r[0]), mx, [v.lower().startswith("active") for v in r[2:6]]))

    def mark(self):
        self.t_mark.append(time.time())

    def stop(self):
        if not self.thread:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml and nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.stop_flag = True
        if self.proc:
            self.proc.terminate()
        self.thread.join(timeout=2)
        # samples inside the timed region; a region shorter than 3 samples falls back to every sample taken while
        # the GPU was under this run's load (warm-up, timed region, e2e)
        window = "timed region"
        sel = [r for r in self.rows if len(self.t_mark) == 2 and self.t_mark[0] <= r[0] <= self.t_mark[1]]
        if len(sel) < 3:
            sel, window = list(self.rows), "warm-up + timed region + e2e (timed region shorter than 3 samples)"
        sm = [r[1] for r in sel]
        mx = [r[2] for r in sel if r[2]]
        reasons = sorted({n for r in sel for n, v in zip(self.NAMES, r[3]) if v})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "window": window, "source": self.source}


def dist_setup(n_gpus):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    return rank, world, local


def barrier_max(ms, world, device="cuda"):
    """max over ranks of a device-timed duration (replicas run independently).  `device` is "cpu" only in the
    gloo test of this helper."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(steps, world, ms_max):
    """BASELINE metric for N independent replicas: rounds all ranks completed / the slowest rank's time."""
    return world * steps / (ms_max * 1e-3)


def sync_all(world):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------------
# CPU oracle on a bounded sample (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_sample(wl, seq_ctx, q_len, n_rows, kv_bits, q_bits, logits, drafts, weights, x_bits, attn_layers=1):
    """Times oracle/ on ONE sequence: `attn_layers` layers of verify attention, one accept/entropy/route,
    and the KV-only prefill of n_rows rows into each drafter.  Returns seconds per part and the outputs."""
    from oracle import accept_route, kv_prefill, verify_attn
    from oracle.paged_kv import PagedKV
    sh = wl.shapes
    n_tok = seq_ctx + q_len
    pages = -(-n_tok // sh.page_size)
    kv = PagedKV(attn_layers, sh.n_kv_heads, sh.head_dim, sh.page_size, pages, 1, pages)
    kv.reserve([n_tok])
    for l in range(attn_layers):
        K, V = kv_bits[l]
        for pg in range(pages):
            cnt = min(sh.page_size, n_tok - pg * sh.page_size)
            kv.k_pool[l, kv.block_table[0, pg], :, :cnt, :] = K[pg * sh.page_size: pg * sh.page_size + cnt].transpose(1, 0, 2)
            kv.v_pool[l, kv.block_table[0, pg], :, :cnt, :] = V[pg * sh.page_size: pg * sh.page_size + cnt].transpose(1, 0, 2)
    kv.seq_len[0] = seq_ctx
    q_indptr = np.array([0, q_len], dtype=np.int32)
    t0 = time.perf_counter()
    outs = [verify_attn.verify_attn(kv, l, q_bits, q_indptr, sh.n_q_heads, 1.0 / np.sqrt(sh.head_dim)) for l in range(attn_layers)]
    t_attn = time.perf_counter() - t0
    t0 = time.perf_counter()
    acc = accept_route.accept_entropy_route(logits, drafts, q_indptr, sh.tau)
    t_acc = time.perf_counter() - t0
    t0 = time.perf_counter()
    for (w_k, w_v) in weights:
        dkv = PagedKV(len(w_k), sh.n_kv_heads, sh.head_dim, sh.page_size, 4, 1, 4)
        d = kv_prefill.Drafter(w_k, w_v, dkv, sh.rope_theta)
        kv_prefill.append_rows(d, [x_bits[:n_rows]])
    t_pre = time.perf_counter() - t0
    return dict(t_attn=t_attn, t_accept=t_acc, t_prefill=t_pre, attn_out=outs, accept=acc)


def gather_sample(rs, b, slot, attn_layers):
    """Copy sequence b's logical K/V (attn_layers layers), its block inputs and the drafter weights to the host."""
    import torch
    sh = rs.sh
    ctx_b = int(rs.seq_len[b].item())
    r0, r1 = int(slot.q_indptr_host[b]), int(slot.q_indptr_host[b + 1])
    n_tok = ctx_b + (r1 - r0)
    pages = rs.block_table[b, : -(-n_tok // sh.page_size)].long()

    def bits(t):
        return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)

    kv_bits = []
    for l in range(attn_layers):
        K = rs.k_pool[l][pages].permute(0, 2, 1, 3).reshape(-1, sh.n_kv_heads, sh.head_dim)[:n_tok]
        V = rs.v_pool[l][pages].permute(0, 2, 1, 3).reshape(-1, sh.n_kv_heads, sh.head_dim)[:n_tok]
        kv_bits.append((bits(K), bits(V)))
    weights = [([bits(w) for w in d.w_k], [bits(w) for w in d.w_v]) for d in rs.drafters.values()]
    return dict(seq_ctx=ctx_b, q_len=r1 - r0, kv_bits=kv_bits, q_bits=bits(slot.q[r0:r1]),
                logits=slot.logits[r0:r1].cpu().numpy(), drafts=slot.drafts[r0:r1].cpu().numpy(),
                weights=weights, x_bits=bits(slot.hidden[r0:r1]))


def round_units(rs, slot):
    """How many single-sequence sample units one round holds (for scaling the oracle sample)."""
    lens = rs.seq_len.cpu().numpy()[: rs.B].astype(np.int64) + slot.q_lens
    return lens


def scale_sample_to_round(t, rs_lens, q_lens, n_layers, b0, n_commit_mean, n0):
    """Seconds the oracle would need for ONE whole round, scaled from the single-sequence sample."""
    attn = t["t_attn"] * n_layers * float(rs_lens.sum()) / float(rs_lens[b0])
    acc = t["t_accept"] * float(q_lens.sum()) / float(q_lens[b0])
    pre = t["t_prefill"] * len(q_lens) * n_commit_mean / max(n0, 1)
    return attn + acc + pre


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on a bounded single-sequence sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = synth.WORKLOADS[WORKLOADS[args.workload]]
    sh = wl.shapes
    g = synth.rng(wl.seed, 1)
    ctx0 = synth.draw_contexts(wl, g)
    gmax = max(wl.gammas)
    q_lens = np.full(wl.batch, gmax + 1, dtype=np.int64)
    b0 = 0
    seq_ctx, q_len = int(ctx0[b0]), int(q_lens[b0])
    n_tok = seq_ctx + q_len
    kv_std = 1.0 / np.sqrt(sh.head_dim)
    kv_bits = [(synth.normal_bf16(g, (n_tok, sh.n_kv_heads, sh.head_dim), kv_std),
                synth.normal_bf16(g, (n_tok, sh.n_kv_heads, sh.head_dim), kv_std))]
    q_bits = synth.normal_bf16(g, (q_len, sh.n_q_heads, sh.head_dim), 1.0)
    u = synth.draw_accept_prefix(g, [gmax], wl.mean_accept)
    logits, drafts, _, _ = synth.make_logits_block(g, [q_len], sh.vocab, sh.logit_sigma, u, [9.0])
    N = sh.n_kv_heads * sh.head_dim
    layers = sh.drafter_layers if len(sh.drafter_layers) == 2 else (sh.drafter_layers[0],) * 2
    weights = [([synth.normal_bf16(g, (sh.hidden, N), 0.02) for _ in range(nl)],
                [synth.normal_bf16(g, (sh.hidden, N), 0.02) for _ in range(nl)]) for nl in layers]
    x_bits = synth.normal_bf16(g, (q_len, sh.hidden), 1.0)
    n_rows = int(u[0]) + 1
    lens = ctx0.astype(np.int64) + q_lens
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        t = oracle_sample(wl, seq_ctx, q_len, n_rows, kv_bits, q_bits, logits, drafts, weights, x_bits)
        if i >= args.warmup:
            times.append((time.perf_counter() - t0, t))
    per_round = float(np.mean([scale_sample_to_round(t, lens, q_lens, sh.n_layers, b0, wl.mean_accept + 1, n_rows) for _, t in times]))
    ms_step = 1e3 * float(np.mean([w for w, _ in times]))
    cores = oracle_cores()
    sample = (f"per step: 1 of {wl.batch} sequences (ctx {seq_ctx}, {q_len} query rows): 1 of {sh.n_layers} attention layers, "
              f"its accept/entropy/route, KV-only prefill of {n_rows} rows into both drafters; scaled to a whole round "
              f"by layers x tokens, rows and sequences")
    value = 1.0 / per_round
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_dict(wl),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def config_dict(wl, world=1):
    """The workload as both arms print it (ours and --impl reference): only what defines the work."""
    sh = wl.shapes
    return {"workload": wl.name, "batch": wl.batch, "ctx": str(wl.ctx), "gammas": list(wl.gammas), "layers": sh.n_layers,
            "vocab": sh.vocab, "backlog_cap": wl.backlog_cap, "switch_prob": wl.switch_prob, "mean_accept": wl.mean_accept,
            "parallelism": "replicas only" if world > 1 else "1 gpu"}


def oracle_cores():
    cores = os.cpu_count()
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        pass
    return cores


def cpu_baseline_and_parity(rs, wl, ctx, wf, n_seq, n_lay):
    """The oracle timed on a bounded sample of slot 0's round (sequences 0..n_seq-1, n_lay attention layers, their
    accept and prefill), which is also the full-size sampled parity check of attention layer 0.  n_seq = B and
    n_lay = L is one WHOLE round, unscaled."""
    import torch
    sh, B, L = rs.sh, rs.B, rs.L
    s0 = rs.slots[0]
    rs.target_kv.reserve(s0.add_tokens, B)                    # pages for the block's own tokens (idempotent)
    wf.wf_verify_attn(ctx, rs.target_kv, 0, s0.q, s0.q_indptr, B, sh.n_q_heads, rs.qmax, rs.sm_scale, s0.attn_out, rs.attn_ws)
    torch.cuda.synchronize()
    lens = round_units(rs, s0)
    tot = {"t_attn": 0.0, "t_accept": 0.0, "t_prefill": 0.0}
    tok = rows_q = rows_p = 0
    worst_rel = worst_abs = 0.0
    for b0 in range(n_seq):
        smp = gather_sample(rs, b0, s0, n_lay)
        n_rows = int(s0.u[b0]) + 1
        t = oracle_sample(wl, smp["seq_ctx"], smp["q_len"], n_rows, smp["kv_bits"], smp["q_bits"], smp["logits"],
                          smp["drafts"], smp["weights"], smp["x_bits"], attn_layers=n_lay)
        for k2 in tot:
            tot[k2] += t[k2]
        tok += int(lens[b0]); rows_q += smp["q_len"]; rows_p += n_rows
        r0, r1 = int(s0.q_indptr_host[b0]), int(s0.q_indptr_host[b0 + 1])
        got = s0.attn_out[r0:r1].float().cpu().numpy().astype(np.float64)     # layer 0 of the launch above
        want = t["attn_out"][0]
        worst_rel = max(worst_rel, float(np.sqrt(((got - want) ** 2).sum() / (want ** 2).sum())))
        worst_abs = max(worst_abs, float(np.abs(got - want).max()))
        if int(t["accept"]["accept_len"][0]) != int(s0.u[b0]):
            raise SystemExit("full-size sampled parity failed: oracle accept_len differs from the planted plan")
    parity = {"attn_rel_l2_layer0_worst": worst_rel, "attn_max_abs_worst": worst_abs, "sequences": n_seq}
    if worst_rel > 5e-3 or worst_abs > 2e-2:
        raise SystemExit(f"full-size sampled parity failed: {parity}")
    whole = n_seq == B and n_lay == L
    if whole:
        per_round = tot["t_attn"] + tot["t_accept"] + tot["t_prefill"]
        sample = (f"ONE WHOLE round, unscaled: all {B} sequence(s) x all {L} attention layers ({tot['t_attn']:.1f} s), accept/entropy/route "
                  f"({tot['t_accept']:.2f} s), KV-only prefill of {rows_p} rows into both drafters ({tot['t_prefill']:.1f} s)")
    else:
        per_round = (tot["t_attn"] * (L / n_lay) * float(lens.sum()) / tok + tot["t_accept"] * float(s0.q_lens.sum()) / rows_q
                     + tot["t_prefill"] * float(np.sum(s0.u + 1)) / rows_p)
        sample = (f"SCALED sample: sequences 0..{n_seq - 1} of {B}: {n_lay} of {L} attention layers ({tot['t_attn']:.1f} s), their "
                  f"accept/entropy/route ({tot['t_accept']:.2f} s), KV-only prefill of {rows_p} rows into both drafters "
                  f"({tot['t_prefill']:.1f} s); scaled to a whole round by layers x tokens, logit rows and committed rows")
    return {"value": 1.0 / per_round, "unit": UNIT, "cores": oracle_cores(), "kind": "oracle", "sample": sample}, parity


def timed_rounds(rs, n, mode, torch):
    """n whole rounds with the given catch-up mode; returns (total ms, catch-up ms, final-token ms inside the catch-up)."""
    mk = lambda: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    ev = [{"attn": mk(), "catchup": mk(), "final": mk()} for _ in range(n)]
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    g0.record()
    for i in range(n):
        rs.run_round(events=ev[i], mode=mode)
    g1.record()
    torch.cuda.synchronize()
    fin = sum(e["final"][0].elapsed_time(e["final"][1]) for e in ev) if (mode != "active" and rs.ft is not None) else 0.0
    return g0.elapsed_time(g1), sum(e["catchup"][0].elapsed_time(e["catchup"][1]) for e in ev), fin


def measure(ctx, wf, key, args, rank, world, local, main):
    """One workload: K timed rounds (device-resident inputs), the e2e leg (host inputs), the catch-up legs, and for the
    main workload the side legs (graph replay, neural router, stochastic acceptance, tree verification)."""
    import torch
    from paper_2606_07710_b200.rounds import RoundState
    wl = synth.WORKLOADS[WORKLOADS[key]]
    sh = wl.shapes
    K, W = (args.steps, max(args.warmup, 3)) if main else (min(args.steps, args.sub_steps), 3)
    e2e_steps = max(1, min(K, args.e2e_steps if main else args.sub_e2e_steps))
    leg_steps = args.slots                                    # one full cycle of the round slots for every catch-up leg
    n_slots = args.slots
    extra = (10 + n_slots + 20) if (main or key == "cfg2") else 0      # tree leg, graph leg
    rs = RoundState(ctx, wl, n_slots=n_slots, n_rounds_max=W + K + e2e_steps + 3 * leg_steps + 4 + extra, host_copies=True)
    B, L = rs.B, rs.L

    # ---- cpu_baseline + full-size sampled parity (rank 0 of a 1-GPU run only) ----
    cpu_baseline, parity = None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        if main:
            cpu_baseline, parity = cpu_baseline_and_parity(rs, wl, ctx, wf, min(B, args.cpu_sample_seqs), min(L, args.cpu_sample_layers))
        elif key == "cfg2":
            cpu_baseline, parity = cpu_baseline_and_parity(rs, wl, ctx, wf, B, L)      # a whole round, no scaling

    # ---- warm-up (the clock sampler starts here so that it is up when the timed region begins) ----
    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(W):
        s = rs.run_round()
    rs.check_plan(s)

    # ---- timed region: K whole rounds, device-resident inputs, CUDA events on the launching stream ----
    evs = [{"attn": (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)),
            "catchup": (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)),
            "final": (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))} for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    attn_bytes = []
    len_host = rs.seq_len.cpu().numpy().astype(np.int64)     # the plan tells us how contexts grow
    launches0 = ctx.launch_count()
    sync_all(world)
    sampler.mark()
    e0.record()
    for i in range(K):
        s = rs.slots[rs.rounds_done % rs.n_slots]
        attn_bytes.append(rs.attn_bytes(s, len_host))
        len_host = len_host + s.u + 1
        rs.run_round(events=evs[i])
    e1.record()
    sync_all(world)
    sampler.mark()
    launches = ctx.launch_count() - launches0
    ms_local = e0.elapsed_time(e1)
    ms = barrier_max(ms_local, world)
    rs.check_plan(s)
    attn_ms = sum(e["attn"][0].elapsed_time(e["attn"][1]) for e in evs)
    # per-round spans from the per-part events (attention start of round i to attention start of round i+1)
    spans = [evs[i]["attn"][0].elapsed_time(evs[i + 1]["attn"][0]) for i in range(K - 1)]
    catch_ms = sum(e["catchup"][0].elapsed_time(e["catchup"][1]) for e in evs)
    final_ms = sum(e["final"][0].elapsed_time(e["final"][1]) for e in evs)
    commits = float(np.mean([np.sum(sl.u + 1) for sl in rs.slots]))
    flips = float(np.mean([np.mean(sl.cur != sl.next) for sl in rs.slots]))

    # ---- e2e: the same rounds through the C-ABI with HOST inputs: H2D of the round's inputs and D2H of
    #      its results inside the timed region (the KV cache is state and stays resident) ----
    host_out = torch.zeros((2, 5, B), dtype=torch.int32).pin_memory()   # accept_len, bonus, route, n_commit, entropy bits; two slots
    h2d = d2h = 0
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all(world)
    # Every step copies its own inputs from pinned host memory and reads its results back inside the timed region;
    # the H2D copy of step i+1 runs on a copy stream while step i computes (the slots are distinct device buffers).
    copy_stream = torch.cuda.Stream()
    d2h_stream = torch.cuda.Stream()
    stage = torch.zeros((2, 5, B), dtype=torch.int32, device="cuda")
    ev_d2h = [None, None]
    main_stream = torch.cuda.current_stream()
    ev_copied = [torch.cuda.Event() for _ in range(rs.n_slots)]
    ev_used = [None] * rs.n_slots

    def issue_copy(k):
        nonlocal h2d
        sl = rs.slots[k]
        with torch.cuda.stream(copy_stream):
            if ev_used[k] is not None:
                copy_stream.wait_event(ev_used[k])           # the slot's previous round has consumed its inputs
            for name, src in sl.host.items():
                getattr(sl, name).copy_(src, non_blocking=True)
                h2d += src.numel() * src.element_size()
            ev_copied[k].record(copy_stream)

    f0.record()
    copy_stream.wait_event(f0)                               # no copy starts before the timed region does
    issue_copy(rs.rounds_done % rs.n_slots)
    for i in range(e2e_steps):
        k = rs.rounds_done % rs.n_slots
        s = rs.slots[k]
        if i + 1 < e2e_steps:
            issue_copy((k + 1) % rs.n_slots)
        main_stream.wait_event(ev_copied[k])
        rs.run_round()
        ev_used[k] = torch.cuda.Event()
        ev_used[k].record(main_stream)
        # the five result vectors of the round in one copy, on a stream of its own: a copy inside the compute stream costs
        # 0.1 ms per round (the next round's first kernel waits for the DMA, measured); round i + 1 does not depend on it
        if ev_d2h[i % 2] is not None:
            main_stream.wait_event(ev_d2h[i % 2])            # the staging slot was read out two rounds ago
        stage[i % 2].copy_(rs.out_all, non_blocking=True)     # 5 x B ints, device to device, in the compute stream
        ev_staged = torch.cuda.Event()
        ev_staged.record(main_stream)
        d2h_stream.wait_event(ev_staged)
        with torch.cuda.stream(d2h_stream):
            host_out[i % 2].copy_(stage[i % 2], non_blocking=True)
            ev_d2h[i % 2] = torch.cuda.Event()
            ev_d2h[i % 2].record(d2h_stream)
        d2h += rs.out_all.numel() * rs.out_all.element_size()
    main_stream.wait_stream(d2h_stream)                       # the timed region ends when the last results are on the host
    f1.record()
    sync_all(world)
    e2e_ms = barrier_max(f0.elapsed_time(f1), world)
    clocks = sampler.stop()
    rs.check_plan(s)

    # ---- catch-up legs, same rounds otherwise (Table 3 at kernel level):
    #      eager  = Lazy Catch-up off: a KV-only prefill into BOTH drafters every round;
    #      active = only the active drafter's own append (reading C22: it stands in for that drafter's forward, which is
    #               drafting cost, not switching cost): lazy - active = what the switch machinery costs per round ----
    for d in rs.drafters.values():                           # flush what the lazy rounds left queued: complete caches
        wf.wf_lazy_catchup_flush(ctx, d.handle, None, B)
    rs.sync_cur()
    lazy_leg_ms, lazy_leg_catch_ms, lazy_leg_final_ms = timed_rounds(rs, leg_steps, "switch", torch)      # the same slots for all three legs
    for d in rs.drafters.values():
        wf.wf_lazy_catchup_flush(ctx, d.handle, None, B)
    rs.rounds_done -= leg_steps
    eager_ms, eager_catch_ms, eager_final_ms = timed_rounds(rs, leg_steps, "eager", torch)
    rs.rounds_done -= leg_steps
    active_ms, active_catch_ms, _ = timed_rounds(rs, leg_steps, "active", torch)
    rs.check_plan(rs.slots[(rs.rounds_done - 1) % rs.n_slots], switched=False)
    rs.sync_cur()
    lazy_us, eager_us, active_us = 1e3 * lazy_leg_catch_ms / leg_steps, 1e3 * eager_catch_ms / leg_steps, 1e3 * active_catch_ms / leg_steps
    final_us = 1e3 * lazy_leg_final_ms / leg_steps
    round_us = 1e3 * ms_local / K

    # ---- (f3) the final backlog token in full, on its own: back-to-back calls for the sequences slot `s` switches to the
    #      AR drafter, and for the whole batch (the weights of the layer are streamed once per call either way) ----
    ft_rec = None
    if rs.ft is not None:
        ft_rec = {"weight_bytes": rs.ft.weight_bytes, "ffn": rs.ft.ffn, "layers": rs.drafters["A"].n_layers}
        sel_sw = s.masks["A"].flush
        for tag, sel, n_tok in (("switching", sel_sw, int(s.masks["A"].flush_host.sum())), ("whole_batch", None, B)):
            for _ in range(3):
                rs.run_final_token(s, sel, 1)
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            t0.record()
            for _ in range(20):
                rs.run_final_token(s, sel, 1)
            t1.record()
            torch.cuda.synchronize()
            us = 1e3 * t0.elapsed_time(t1) / 20
            # algorithmic bytes of a call: the layer's four matrices once + the drafter-cache K/V of the selected sequences
            # (one query row each over its whole cached context, every drafter layer)
            dA = rs.drafters["A"]
            lens = dA.seq_len.cpu().numpy().astype(np.int64)
            picked = lens if sel is None else lens[s.masks["A"].flush_host.astype(bool)]
            kv_bytes = int(picked.sum()) * sh.n_kv_heads * sh.head_dim * 2 * 2 * dA.n_layers
            tot = rs.ft.weight_bytes + kv_bytes
            ft_rec[tag] = {"tokens": n_tok, "us_per_call": us, "kv_bytes": kv_bytes,
                           "weight_gbs": rs.ft.weight_bytes / (us * 1e-6) / 1e9 if n_tok else None,
                           "hbm_gbs": tot / (us * 1e-6) / 1e9 if n_tok else None}

    peak, peak_src = measured_peaks()
    if ft_rec:
        for tag in ("switching", "whole_batch"):
            g_ = ft_rec[tag]["hbm_gbs"]
            ft_rec[tag]["frac_of_hbm_peak"] = g_ / peak if g_ else None
        ft_rec["note"] = ("wf_final_token_full for the AR drafter (one transformer layer, PAPER.md:231): Q/O/up/down weight streams "
                          "(weight_bytes) + one-row attention over the drafter cache (kv_bytes of the selected sequences); hbm_gbs and "
                          "frac_of_hbm_peak count both; 'switching' = the sequences the "
                          "last timed slot switches to the AR drafter, 'whole_batch' = every sequence; back-to-back calls")
    avg_launch_ms = attn_ms / (K * L)
    achieved = float(np.mean(attn_bytes)) / (avg_launch_ms * 1e-3) / 1e9
    traffic, traffic_src = NCU_TRAFFIC.get(key, (None, None))
    if main and args.traffic_bytes is not None:
        traffic, traffic_src = args.traffic_bytes, "--traffic-bytes"
    rec = {
        "value": whole_job_value(K, world, ms), "unit": UNIT, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "ms_per_step_median": float(np.median(spans)) if spans else ms / K,
        "config": config_dict(wl, world),
        "run_notes": {"slots": rs.n_slots, "realised_switch_rate": flips, "attn_early_kv": int(args.attn_early),
                      "l2": f"inputs larger than L2: {np.mean(attn_bytes) / 1e6:.0f} MB of KV per attention launch, distinct per layer",
                      "catchup": "lazy: one wf_switch_round per round (both drafters, masks derived on the device from route), then "
                                 "wf_final_token_full for the sequences that switched to the AR drafter"},
        "committed_tokens_per_s": world * commits * K / (ms * 1e-3),
        "kv_read_gbs": achieved,
        "attn_share_of_round": attn_ms / ms_local,
        "catchup_us_per_round": lazy_us,
        "catchup_share_of_round": catch_ms / ms_local,
        "catchup": {"lazy_us_per_round": lazy_us, "eager_us_per_round": eager_us, "active_append_us_per_round": active_us,
                    "final_token_us_per_round": final_us, "flush_us_per_round": lazy_us - final_us,
                    "eager_kv_us_per_round": eager_us - 1e3 * eager_final_ms / leg_steps,
                    "switch_us_per_round": lazy_us - active_us, "share_of_round": lazy_us / round_us,
                    "flush_share_of_round": (lazy_us - final_us) / round_us,
                    "final_token_share_of_round": final_us / round_us,
                    "switch_share_of_round": (lazy_us - active_us) / round_us, "eager_share_of_round": eager_catch_ms / eager_ms,
                    "eager_rounds_per_s": leg_steps / (eager_ms * 1e-3), "lazy_rounds_per_s": leg_steps / (lazy_leg_ms * 1e-3),
                    "leg_steps": leg_steps,
                    "note": "three legs over the same full cycle of round slots; lazy = wf_switch_round (+ final token); eager = KV-only prefill into both drafters every round "
                            "(Lazy Catch-up off, PAPER.md Table 3 baseline); active_append = only the active drafter's own append "
                            "(reading C22: drafting cost, not switching cost); switch = lazy - active_append (derived); "
                            "final_token = wf_final_token_full for the sequences that switched to the AR drafter (PAPER.md:119), "
                            "inside lazy and eager alike; flush = lazy - final_token is what Lazy Catch-up costs per round (rows (c) + (d) of "
                            "north_star: flush_share_of_round is the figure its 7 % bar is about; share_of_round also counts f3) and "
                            "eager_kv = eager - its final token what the naive scheme costs (PAPER.md Table 3)"},
        "roofline": {"bound": "hbm", "kernel": "wf_verify_attn_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "peak_source": peak_src, "traffic": traffic, "traffic_source": traffic_src,
                     "algorithmic_bytes_per_launch": float(np.mean(attn_bytes)), "avg_launch_us": 1e3 * avg_launch_ms},
        "e2e": {"value": world * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d // e2e_steps,
                "d2h_bytes_per_step": d2h // e2e_steps, "steps": e2e_steps,
                "overlap": "H2D of step i+1 on a copy stream while step i computes, D2H of step i on a third stream; every copy is inside the timed region"},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if ft_rec:
        rec["final_token"] = ft_rec
    if cpu_baseline:
        rec["cpu_baseline"] = cpu_baseline
        rec["parity_sample"] = parity
    if main:
        rec.update(side_legs(rs, ctx, wf, wl, args, s, peak, torch))
    elif key == "cfg2":                                      # batch 1 is launch-paced: the graph replay is its B200-native form
        rec.update(side_legs(rs, ctx, wf, wl, args, s, peak, torch, only_graph=True))
    rs.close()
    return rec


def side_legs(rs, ctx, wf, wl, args, s, peak, torch, only_graph=False):
    """Legs timed on their own after the headline region: graph replay, neural router, stochastic acceptance, tree verify."""
    sh, B, L = rs.sh, rs.B, rs.L
    out = {}
    # ---- the same round replayed from CUDA graphs (SURVEY.md §8(d) timing protocol): one graph per round slot, captured
    #      from the very calls above (every argument is a device pointer or a constant; lengths live on the device) ----
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        graphs = []
        for _ in range(rs.n_slots):
            gph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gph, stream=side):
                rs.run_round()
            graphs.append(gph)
        torch.cuda.synchronize()
        g_steps = 20
        for i in range(rs.n_slots):
            graphs[i].replay()
        torch.cuda.synchronize()
        h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        h0.record()
        for i in range(g_steps):
            graphs[i % rs.n_slots].replay()
        h1.record()
        torch.cuda.synchronize()
        rs.check_plan(rs.slots[(rs.rounds_done + g_steps - 1) % rs.n_slots])
        rs.rounds_done += g_steps                            # the replays advanced the device state by g_steps rounds
        out["graph_replay"] = {"rounds_per_s": g_steps / (h0.elapsed_time(h1) * 1e-3), "steps": g_steps,
                               "note": "whole round replayed from one CUDA graph per round slot, captured from the same C-ABI calls"}
        del graphs
    except Exception as e:                                   # capture is optional evidence, never the headline
        out["graph_replay"] = {"error": f"{type(e).__name__}: {e}"[:200]}
        torch.cuda.synchronize()

    if only_graph:
        return out
    # ---- WhiFlash-Neural router, timed on its own: the round above uses the entropy policy ----
    n0, n1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        rs.run_neural_route(s)
    torch.cuda.synchronize()
    n0.record()
    for _ in range(20):
        rs.run_neural_route(s)
    n1.record()
    torch.cuda.synchronize()
    out["neural_router"] = {"us_per_call": 1e3 * n0.elapsed_time(n1) / 20, "params": rs.nr.d * rs.nr.m + 2 * rs.nr.m + 1, "batch": B,
                            "note": "WhiFlash-Neural policy (d -> d/8 -> GELU -> 1), back-to-back calls, not part of the round"}

    # ---- stochastic acceptance next to the greedy sweep, both on the last slot's logits, cache
    #      length untouched (target_kv = NULL): one sweep over the logits + the per-sequence inverse-CDF draw ----
    gsmp = torch.Generator(device="cuda")
    gsmp.manual_seed(wl.seed)
    u_acc = torch.rand(s.sum_q, dtype=torch.float32, device="cuda", generator=gsmp)
    u_smp = torch.rand(B, dtype=torch.float32, device="cuda", generator=gsmp)
    tok_out = torch.zeros(B, dtype=torch.int32, device="cuda")
    acc_us = {}
    # a drafter distribution per row for the full-q variant: softmax of a perturbed copy of the logits (input construction)
    q_full = torch.softmax(s.logits / 0.8 * 0.9 + torch.randn(s.logits.shape, device="cuda", generator=gsmp), dim=1)
    scratch = {k: torch.zeros_like(v) for k, v in rs.out.items()}          # the round's own outputs stay untouched
    ent = torch.zeros_like(rs.entropy)
    for mode in ("greedy", "sample", "sample_full_q"):
        def call():
            o = scratch
            if mode == "sample_full_q":
                wf.wf_accept_sample_entropy_route(ctx, s.logits, sh.vocab, s.drafts, s.q_indptr, B, rs.qmax, 0.8, q_full, u_acc, u_smp,
                                                  rs.tau, True, o["accept_len"], tok_out, ent, o["route"], o["n_commit"],
                                                  None, rs.acc_ws)
            elif mode == "greedy":
                wf.wf_accept_entropy_route(ctx, s.logits, sh.vocab, s.drafts, s.q_indptr, B, rs.qmax, rs.tau, True, o["accept_len"],
                                           tok_out, ent, o["route"], o["n_commit"], None, rs.acc_ws)
            else:
                wf.wf_accept_sample_entropy_route(ctx, s.logits, sh.vocab, s.drafts, s.q_indptr, B, rs.qmax, 0.8, None, u_acc, u_smp,
                                                  rs.tau, True, o["accept_len"], tok_out, ent, o["route"], o["n_commit"],
                                                  None, rs.acc_ws)
        for _ in range(3):
            call()
        torch.cuda.synchronize()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        for _ in range(20):
            call()
        a1.record()
        torch.cuda.synchronize()
        acc_us[mode] = 1e3 * a0.elapsed_time(a1) / 20
    logit_bytes = float(s.sum_q) * sh.vocab * 4
    del q_full
    out["stochastic_accept"] = {"us_per_call": acc_us["sample"], "greedy_us_per_call": acc_us["greedy"],
                                "full_q_us_per_call": acc_us["sample_full_q"], "temperature": 0.8,
                                "logits_gbs": logit_bytes / (acc_us["sample"] * 1e-6) / 1e9,
                                "greedy_logits_gbs": logit_bytes / (acc_us["greedy"] * 1e-6) / 1e9,
                                "greedy_frac_of_hbm_peak": logit_bytes / (acc_us["greedy"] * 1e-6) / 1e9 / peak,
                                "note": "speculative sampling (one-hot drafter, uniforms as inputs): same sweep over the "
                                        "logits plus one inverse-CDF draw per sequence; back-to-back calls on the "
                                        "logits of the last slot, not part of the round"}

    # ---- tree verification round, timed on its own: every sequence brings a 60-node draft tree
    #      (PAPER.md:317); masks + L x tree attention + acceptance walk + path compaction ----
    if not args.no_tree:
        tsl = rs.make_tree_slot(60)
        tree_steps = 6
        ev_t = [{"attn": (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))} for _ in range(tree_steps)]
        for _ in range(2):
            rs.run_tree_round(tsl)
        rs.check_tree_plan(tsl)
        t_len = rs.seq_len.cpu().numpy().astype(np.int64)
        t_commit = np.array([len(p) for p in tsl.paths], dtype=np.int64)
        t_bytes = []
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for i in range(tree_steps):
            t_bytes.append(int((t_len + 60).sum()) * sh.n_kv_heads * sh.head_dim * 2 * 2)
            t_len = t_len + t_commit
            rs.run_tree_round(tsl, events=ev_t[i])
        t1.record()
        rs.check_tree_plan(tsl)
        tree_ms = t0.elapsed_time(t1)
        tree_attn_ms = sum(e["attn"][0].elapsed_time(e["attn"][1]) for e in ev_t)
        gbs = float(np.mean(t_bytes)) / (tree_attn_ms / (tree_steps * L) * 1e-3) / 1e9
        out["tree_verify"] = {"rounds_per_s": tree_steps / (tree_ms * 1e-3), "ms_per_round": tree_ms / tree_steps, "steps": tree_steps,
                              "nodes": 60, "attn_us_per_launch": 1e3 * tree_attn_ms / (tree_steps * L), "kv_read_gbs": gbs,
                              "frac_of_hbm_peak": gbs / peak, "committed_tokens_per_round": float(t_commit.sum()),
                              "note": "all sequences AR-routed with depth-8 / top-k-10 / 60-node trees (PAPER.md:317); 240 query rows per "
                                      "kv head = two 128-row query tiles (UMMA M = 128) that stream the same K/V (HBM once, L2 for the second)"}
    return out


def run_ours(args):
    import torch
    rank, world, local = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    from paper_2606_07710_b200 import binding as wf          # raises if libwhiflash.so is missing: no fallback
    ctx = wf.Ctx(local)
    # the round is reserve -> L x attention -> accept -> switch -> final token: no kernel that precedes an attention launch
    # writes lengths, old block-table entries or cached rows below the cached length (the promise of wf_ctx_set_attn_early_kv)
    ctx.set_attn_early_kv(args.attn_early)
    if args.attn_cluster != -1:
        ctx.set_attn_cluster(args.attn_cluster)
    rec = measure(ctx, wf, args.workload, args, rank, world, local, main=True)
    per_config = {}
    for key in [k for k in args.sub_workloads.split(",") if k and k != args.workload]:
        torch.cuda.empty_cache()
        sub = measure(ctx, wf, key, args, rank, world, local, main=False)
        keep = ("value", "unit", "steps", "ms_per_step", "kv_read_gbs", "attn_share_of_round", "catchup", "final_token", "roofline", "e2e",
                "clocks", "cpu_baseline", "parity_sample", "committed_tokens_per_s", "gpu_launches", "graph_replay")
        per_config[key] = {k: sub[k] for k in keep if k in sub}
        per_config[key]["workload"] = sub["config"]["workload"]
        per_config[key]["realised_switch_rate"] = sub["run_notes"]["realised_switch_rate"]
    if rank == 0:
        line = {"metric": METRIC, "value": rec.pop("value"), "unit": rec.pop("unit"), "n_gpus": world, "steps": rec.pop("steps"),
                "warmup": rec.pop("warmup"), "ms_per_step": rec.pop("ms_per_step"), "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic"}
        line.update(rec)
        if per_config:
            line["per_config"] = per_config
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=60)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS),
                    help="the headline workload: cfg5 = BASELINE.json configs[4], the largest single-GPU config")
    ap.add_argument("--sub-workloads", default="cfg2,cfg3,cfg4",
                    help="comma-separated workloads reported as compact per_config sub-records of the same line ('' = none)")
    ap.add_argument("--sub-steps", type=int, default=30)
    ap.add_argument("--sub-e2e-steps", type=int, default=30)
    ap.add_argument("--slots", type=int, default=16, help="round slots of the cyclic schedule (distinct inputs and plans)")
    ap.add_argument("--e2e-steps", type=int, default=30)
    ap.add_argument("--attn-early", type=int, default=1, choices=[0, 1],
                    help="wf_ctx_set_attn_early_kv: attention launches stream the cached K/V ahead of the dependency wait")
    ap.add_argument("--attn-cluster", type=int, default=-1, help="wf_ctx_set_attn_cluster (tuning hook; -1 = automatic)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-tree", action="store_true", help="skip the tree-verification leg (SURVEY.md §8(f) f2)")
    ap.add_argument("--cpu-sample-seqs", type=int, default=8)
    ap.add_argument("--cpu-sample-layers", type=int, default=16)
    ap.add_argument("--traffic-bytes", type=float, default=None,
                    help="dram bytes per attention launch; default: the committed ncu --set full capture for the workload")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
