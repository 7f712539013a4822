#!/usr/bin/env python
"""bench.py -- codec tokens/s of the MAPL boundary codec on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mapl|reference] [--workload c1|c2|c3]

One "step" = one pass of the whole hot path over one batch of synthetic input: for every stage
boundary of the workload, mapl_encode -> mapl_decode (forward order), then mapl_codec_backward in
reverse order (full backward: H given, dH and dA produced, dB off as in the paper), plus one
mapl_stiefel_step per boundary when the workload says so (c3).  A codec token = one token crossing
one boundary through all three calls; value = N * n_boundaries * n_gpus * K / time.

Timing: W >= 3 warm-up steps, then exactly K steps between barrier + synchronize, CUDA events on
the launching stream, max over ranks.  The K steps replay one CUDA graph of the step (the calls are
launch-bound from Python otherwise).  Every boundary has its own buffers; the per-step working set
(hundreds of MB) exceeds the 126 MB L2, so no flush is needed between iterations.

Prints ONE JSON line (rank 0).  Multi-GPU: one process per GPU under torchrun, independent
micro-batches per rank (weak scaling), no data-path collective.
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "codec tokens/s (enc+dec fwd+bwd, proj+RVQ+anchor)"
UNIT = "tokens/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return dict(hbm=float(j["hbm_gbs"]), bf16=float(j["bf16_tflops"]),
                    bf16_sustained=float(j.get("bf16_tflops_sustained", j["bf16_tflops"])), src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, src="fallback")


# ---------------------------------------------------------------- workload description

def workload(name: str):
    from paper_2606_05484_b200 import inputs as I
    cfg = I.CONFIGS[name]
    desc = (f"{name}: N={cfg.n_tokens} d={cfg.d} r={cfg.r} L={cfg.rvq_levels} K={cfg.rvq_k} V={cfg.vocab} "
            f"ra={cfg.anchor_rank} {cfg.act_dtype}, {cfg.n_boundaries} boundaries, enc+dec+bwd(dH,dA; dB off)"
            + (" + stiefel step/boundary" if name == "c3" else ""))
    return cfg, desc


def alg_bytes_per_token(cfg):
    """what the method itself must move per token per boundary."""
    s = 2 if cfg.act_dtype == "bf16" else 4
    d, r, L = cfg.d, cfg.r, cfg.rvq_levels
    payload = r * s if L == 0 else 4 * L
    enc = d * s + payload
    dec = payload + 4 + d * s
    bwd = 3 * d * s + payload + r * s + 4      # g, H read; dH written; payload (Z or codes) read; gz written; tok
    return dict(encode=enc, decode=dec, backward=bwd)


def alg_flops_per_token(cfg):
    d, r, ra, L, K = cfg.d, cfg.r, cfg.anchor_rank, cfg.rvq_levels, cfg.rvq_k
    return dict(encode=2 * d * r + L * 2 * K * r, decode=2 * (r + ra) * d, backward=8 * d * r + 2 * d * ra)


# ---------------------------------------------------------------- clocks sampler

class ClockSampler:
    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {getattr(nv, n): n[len("nvmlClocksEventReason"):] for n in dir(nv)
                 if n.startswith("nvmlClocksEventReason") and isinstance(getattr(nv, n), int)} or \
                {getattr(nv, n): n[len("nvmlClocksThrottleReason"):] for n in dir(nv)
                 if n.startswith("nvmlClocksThrottleReason") and isinstance(getattr(nv, n), int)}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if bit and (mask & bit) and nm not in ("None", "All"):
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv:
            self._t = threading.Thread(target=self._loop, daemon=True)
            self._t.start()

    def stop(self):
        self._stop.set()
        if self._t:
            self._t.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": []}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


# ---------------------------------------------------------------- multi-rank host logic (replicas only)

def boundary_stream(b: int, rank: int) -> int:
    """Seed stream of boundary b on rank `rank`: every rank draws its own micro-batches (weak scaling,
    no data-path collective)."""
    return b + 16 * rank


def max_over_ranks(values, world: int, device):
    """Element-wise MAX over the ranks of device-measured times (the job is as slow as its slowest
    replica).  The only collective of the multi-GPU run; covered on CPU by the gloo test."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_tokens_per_second(tokens_per_rank_step: int, world: int, steps: int, ms: float) -> float:
    """Whole-job aggregate: all ranks' tokens over the slowest rank's time."""
    return tokens_per_rank_step * world * steps / (ms * 1e-3)


# ---------------------------------------------------------------- the CUDA arm

class Boundary:
    """device buffers of one stage boundary (own copies: nothing is shared between boundaries)"""

    def __init__(self, cfg, b, rank, torch, mb, I, host=False):
        bi = I.make_boundary(cfg, boundary_stream(b, rank))
        self.cfg = cfg
        act = torch.bfloat16 if cfg.act_dtype == "bf16" else torch.float32

        def dev(s):
            if isinstance(s, np.ndarray):
                return torch.from_numpy(s.copy()).cuda()
            t = torch.from_numpy(s.data.copy())
            return (t.view(torch.bfloat16) if s.dtype == "bf16" else t).cuda()

        def pin(s):
            if isinstance(s, np.ndarray):
                return torch.from_numpy(s.copy()).pin_memory()
            t = torch.from_numpy(s.data.copy())
            return (t.view(torch.bfloat16) if s.dtype == "bf16" else t).pin_memory()

        N, d, r, L = cfg.n_tokens, cfg.d, cfg.r, cfg.rvq_levels
        self.desc = mb.make_desc(N, d, r, act, L, cfg.rvq_k if L else 0, cfg.vocab, cfg.anchor_rank)
        self.H, self.g, self.tok = dev(bi.H), dev(bi.g), dev(bi.tok)
        self.U, self.A, self.B = dev(bi.U), dev(bi.A), dev(bi.B)
        self.C = dev(bi.C) if bi.C is not None else None
        e = lambda *shape, dt=act: torch.empty(shape, dtype=dt, device="cuda")
        self.Zq = e(N, r) if L == 0 else None
        self.codes = e(N, L, dt=torch.int32) if L > 0 else None
        self.Hhat, self.gz, self.dH = e(N, d), e(N, r), e(N, d)
        self.dU = e(d, r, dt=torch.float32)
        self.dA = e(cfg.vocab, cfg.anchor_rank, dt=torch.float32)
        self.ws = mb.alloc_workspace(mb.mapl_workspace_bytes(self.desc))
        # prepared bf16 parameter pack (include/mapl.h), shared by the three codec calls of a boundary.
        # Workloads whose step updates U (c3: Stiefel step) rebuild it inside the timed region, once
        # per boundary per step; where the parameters are constant across steps (c1, c2) it is built
        # once, before the timed region, like any weight-layout preparation.
        nb = mb.mapl_param_pack_bytes(self.desc)
        self.pack = mb.alloc_workspace(nb) if nb else None
        if self.pack is not None:
            self.desc.param_pack = self.pack.data_ptr()
        if host:
            self.hH, self.hg, self.htok = pin(bi.H), pin(bi.g), pin(bi.tok)
            ph = lambda t: torch.empty(t.shape, dtype=t.dtype).pin_memory()
            self.o_payload = ph(self.Zq if L == 0 else self.codes)
            self.o_Hhat, self.o_gz, self.o_dH, self.o_dU = ph(self.Hhat), ph(self.gz), ph(self.dH), ph(self.dU)


def make_step(bs, mb, stiefel=None):
    for b in bs:
        if b.pack is not None:
            mb.mapl_pack_params(b.desc, b.U, b.B, b.C, b.pack)

    def fwd(b):
        if b.pack is not None and stiefel is not None:
            mb.mapl_pack_params(b.desc, b.U, None, None, b.pack)    # U changed (Stiefel step); B and the codebooks did not
        mb.mapl_encode(b.desc, b.H, b.U, b.C, b.Zq, b.codes, b.ws)
        mb.mapl_decode(b.desc, b.Zq, b.codes, b.U, b.C, b.tok, b.A, b.B, b.Hhat, b.ws)

    def bwd(b):
        mb.mapl_codec_backward(b.desc, b.g, b.H, b.Zq, b.codes, b.U, b.C, b.tok, b.A, b.B, b.gz, b.dU, b.dA,
                               None, b.dH, False, b.ws)

    def step():
        for b in bs:
            fwd(b)
        for b in reversed(bs):
            bwd(b)
        if stiefel is not None:
            stiefel()
    return step


def run_mapl(args):
    import torch
    import torch.distributed as dist
    from paper_2606_05484_b200 import binding as mb
    from paper_2606_05484_b200 import inputs as I

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU path"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg, wdesc = workload(args.workload)
    if args.tokens:
        cfg = cfg.with_tokens(args.tokens)
    nb = cfg.n_boundaries
    bs = [Boundary(cfg, b, rank, torch, mb, I, host=True) for b in range(nb)]
    lib = mb.raw_lib()

    stiefel = None
    if args.workload == "c3":       # configs[3]: "plus a Stiefel step per boundary" (G = dU / N, S12)
        # the nb projectors live in one [nb, d, r] tensor (and their gradients likewise), so the per-boundary
        # Stiefel steps of a training step are ONE batched mapl_stiefel_step call (batch = nb)
        st_ws = mb.alloc_workspace(mb.mapl_stiefel_workspace_bytes(cfg.d, cfg.r, nb))
        Uall = torch.stack([b.U for b in bs]).contiguous()
        dUall = torch.empty_like(Uall)
        Gall = torch.empty_like(Uall)
        for i, b in enumerate(bs):
            b.U, b.dU = Uall[i], dUall[i]

        def stiefel():
            torch.mul(dUall, 1.0 / cfg.n_tokens, out=Gall)
            mb.mapl_stiefel_step(Uall, Gall, 1e-2, mb.MAPL_RETRACT_NS, 5, None, st_ws)
    step = make_step(bs, mb, stiefel)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        for _ in range(max(3, args.warmup)):
            step()
        stream.synchronize()
        # count our launches in one step
        lib.mapl_profile_reset()
        step()
        stream.synchronize()
        launches_per_step = 0
        for kid in range(lib.mapl_profile_kernel_count()):
            n = C.c_longlong(0)
            lib.mapl_profile_read(kid, C.byref(n), None, None)
            launches_per_step += n.value
        # capture the step once, replay K times
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            step()
        for _ in range(3):
            graph.replay()
        stream.synchronize()

        sampler = ClockSampler(local)
        barrier()
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            graph.replay()
        e1.record(stream)
        stream.synchronize()
        barrier()
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1)

        # ---- per-call times: one CUDA graph per entry point (all boundaries, 4 repetitions), replayed 10 times.
        # Graph replay keeps the programmatic-dependent-launch overlap the step has, unlike the
        # event-bracketed eager pass below, whose per-kernel times include launch latency.
        def graph_us(fn, reps=4, replays=10):
            for b in bs:
                fn(b)
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                for _ in range(reps):
                    for b in bs:
                        fn(b)
            g.replay()
            stream.synchronize()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record(stream)
            for _ in range(replays):
                g.replay()
            c1.record(stream)
            stream.synchronize()
            return 1e3 * c0.elapsed_time(c1) / (replays * reps * len(bs))
        calls_us = {
            "mapl_encode": graph_us(lambda b: mb.mapl_encode(b.desc, b.H, b.U, b.C, b.Zq, b.codes, b.ws)),
            "mapl_decode": graph_us(lambda b: mb.mapl_decode(b.desc, b.Zq, b.codes, b.U, b.C, b.tok, b.A, b.B, b.Hhat, b.ws)),
            "mapl_codec_backward": graph_us(lambda b: mb.mapl_codec_backward(
                b.desc, b.g, b.H, b.Zq, b.codes, b.U, b.C, b.tok, b.A, b.B, b.gz, b.dU, b.dA, None, b.dH, False, b.ws)),
            # the receiver's share alone (H == NULL: gz, dA and the decode-side term of dU; no dH), reported beside the headline
            "mapl_codec_backward_decode_side": graph_us(lambda b: mb.mapl_codec_backward(
                b.desc, b.g, None, b.Zq, b.codes, b.U, b.C, b.tok, b.A, b.B, b.gz, b.dU, b.dA, None, None, False, b.ws)),
        }

        # ---- per-kernel timing pass (same K steps, eager launches, event pair around every kernel)
        lib.mapl_profile_reset()
        lib.mapl_profile_enable(1)
        for _ in range(args.steps):
            step()
        stream.synchronize()
        lib.mapl_profile_enable(0)
        kern = {}
        for kid in range(lib.mapl_profile_kernel_count()):
            n, nt, tms = C.c_longlong(0), C.c_longlong(0), C.c_double(0)
            lib.mapl_profile_read(kid, C.byref(n), C.byref(nt), C.byref(tms))
            if nt.value:
                kern[lib.mapl_profile_kernel_name(kid).decode()] = dict(launches=nt.value, ms=tms.value)

        # ---- end to end: pinned host inputs -> device, the three calls, results -> pinned host.
        # Three streams, as a user of the library would drive it: the uploads of step i+1 run while the
        # results of step i are downloaded (PCIe is full duplex); the codec calls of a step wait for
        # its uploads and for the previous step's downloads (they overwrite the same device buffers).
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        ev_in, ev_done, ev_out = torch.cuda.Event(), torch.cuda.Event(), torch.cuda.Event()
        ev_done.record(stream)
        ev_out.record(s_out)

        def e2e_step():
            s_in.wait_event(ev_done)                       # the previous step no longer reads H, tok, g
            with torch.cuda.stream(s_in):
                for b in bs:
                    b.H.copy_(b.hH, non_blocking=True)
                    b.tok.copy_(b.htok, non_blocking=True)
                    b.g.copy_(b.hg, non_blocking=True)
                ev_in.record(s_in)
            stream.wait_event(ev_in)
            stream.wait_event(ev_out)                      # the previous results have left the device
            step()
            ev_done.record(stream)
            s_out.wait_event(ev_done)
            with torch.cuda.stream(s_out):
                for b in bs:
                    b.o_payload.copy_(b.Zq if b.Zq is not None else b.codes, non_blocking=True)
                    b.o_Hhat.copy_(b.Hhat, non_blocking=True)
                    b.o_gz.copy_(b.gz, non_blocking=True)
                    b.o_dH.copy_(b.dH, non_blocking=True)
                    b.o_dU.copy_(b.dU, non_blocking=True)
                ev_out.record(s_out)
        nbytes = lambda t: t.numel() * t.element_size()
        h2d = sum(nbytes(b.hH) + nbytes(b.htok) + nbytes(b.hg) for b in bs)
        d2h = sum(nbytes(b.o_payload) + nbytes(b.o_Hhat) + nbytes(b.o_gz) + nbytes(b.o_dH) + nbytes(b.o_dU) for b in bs)
        e2e_steps = max(1, min(args.steps, 20))
        for _ in range(2):
            e2e_step()
        stream.wait_event(ev_out)
        barrier()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(stream)
        for _ in range(e2e_steps):
            e2e_step()
        stream.wait_event(ev_out)                          # the last results are in host memory
        f1.record(stream)
        stream.synchronize()
        barrier()
        e2e_ms = f0.elapsed_time(f1)

    ms, e2e_ms = max_over_ranks([ms, e2e_ms], world, "cuda")
    value = job_tokens_per_second(cfg.n_tokens * nb, world, args.steps, ms)
    e2e_value = job_tokens_per_second(cfg.n_tokens * nb, world, e2e_steps, e2e_ms)

    # ---- roofline of the dominant kernel (largest share of the timed per-kernel pass)
    peaks = _peaks()
    roof = None
    if kern:
        top = max(kern, key=lambda k: kern[k]["ms"])
        total = sum(v["ms"] for v in kern.values())
        roof = roofline_for(top, kern[top], cfg, peaks, total)
        roof["kernels"] = {k: {"launches": v["launches"], "avg_us": round(1e3 * v["ms"] / v["launches"], 2),
                               "share": round(v["ms"] / total, 3)} for k, v in sorted(kern.items(), key=lambda kv: -kv[1]["ms"])}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.act_dtype, "data": "synthetic",
        "config": {"workload": wdesc, "l2": "distinct buffers per boundary; per-step working set > 126 MB L2, no flush",
                   "launch": "one CUDA graph of the step, replayed K times",
                   "param_pack": ("rebuilt per boundary per step (U changes every step)" if stiefel is not None
                                  else "built once before the timed region (parameters constant across steps)"), "parallelism": f"replicas x{world}"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "note": "pinned host H,tok,g -> device; payload,Hhat,gz,dH,dU -> pinned host; uploads of step i+1 overlap downloads of step i (3 streams)"},
        "roofline_step": roofline_step(cfg, peaks, ms / args.steps, nb, calls_us),
        "gpu_launches": launches_per_step * args.steps,
        "calls_us": {k: round(v, 2) for k, v in calls_us.items()},
        "roofline": roof,
    }
    if rank == 0 and world == 1 and not args.no_stiefel:
        out["stiefel"] = stiefel_sweep(torch, mb, I, stream, track_steps=args.track_steps)
    if rank == 0 and world == 1 and not args.no_stiefel:
        out["centering"] = centering_times(torch, mb, bs[0], cfg, stream)
    if rank == 0:
        if not args.no_cpu_baseline and world >= 1:
            out["cpu_baseline"] = cpu_baseline(cfg, budget_s=args.cpu_budget)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def _stiefel_track(torch, mb, s, r, retr, ws, stream, n_steps):
    """configs[4]: `n_steps` consecutive steps with ||U^T U - I||_F tracked -- on the device by the library every step
    (info_out, fp32 Gram: its maximum over the run) and in fp64 (torch) at steps 1, 2, 10, 100, 500, 1000 -- for the
    fixed seeded gradient and for a fresh Gaussian gradient every step (reading S13; drawn by torch's seeded device
    generator: an input, not part of the method).  Maximum over the 3 projectors."""
    marks = [m for m in (1, 2, 10, 100, 500, 1000) if m <= n_steps]
    eye = torch.eye(r, device="cuda", dtype=torch.float64)
    res = {}
    for variant in ("fixed_G", "fresh_G"):
        U = torch.from_numpy(s.U.data.copy()).cuda()
        G = torch.from_numpy(s.G.data.copy()).cuda()
        info = torch.zeros(s.batch, 2, device="cuda", dtype=torch.float32)
        log = torch.zeros(n_steps, device="cuda", dtype=torch.float32)
        gen = torch.Generator(device="cuda")
        gen.manual_seed(260605484 + r)
        mb.mapl_stiefel_step(U, G, 1e-2, retr, 5, info, ws)
        stream.synchronize()
        U.copy_(torch.from_numpy(s.U.data.copy()))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            mb.mapl_stiefel_step(U, G, 1e-2, retr, 5, info, ws)
        U.copy_(torch.from_numpy(s.U.data.copy()))
        at = {}
        for t in range(1, n_steps + 1):
            if variant == "fresh_G":
                G.normal_(generator=gen)
            g.replay()
            log[t - 1] = info[:, 1].max()
            if t in marks:
                Uh = U.double()
                at[str(t)] = float(f"{float(max(torch.linalg.matrix_norm(Uh[b].T @ Uh[b] - eye) for b in range(s.batch))):.2e}")
        stream.synchronize()
        res[variant] = {"residual_fp64_at_step": at, "max_device_residual": float(f"{float(log.max()):.2e}"), "steps": n_steps}
    return res


def stiefel_sweep(torch, mb, I, stream, reps=10, track_steps=1000):
    """BASELINE.json configs[4] beside the codec metric: Stiefel steps/s for the 3 projectors of d=2048,
    r in {64,128,256,512}, QR (CholeskyQR2) and 5 Newton-Schulz iterations; one CUDA graph per variant.
    A step = one mapl_stiefel_step call over the batch of 3; projector-steps/s = 3 x that.
    `track`: the variant repeated for track_steps steps from the seeded start, with the orthogonality residual
    tracked (see _stiefel_track)."""
    out = {}
    with torch.cuda.stream(stream):
        for r in (64, 128, 256, 512):
            s = I.make_stiefel(r)
            ws = mb.alloc_workspace(mb.mapl_stiefel_workspace_bytes(s.d, r, s.batch))
            for retr, tag in ((mb.MAPL_RETRACT_NS, "ns5"), (mb.MAPL_RETRACT_QR, "qr")):
                U = torch.from_numpy(s.U.data.copy()).cuda()
                G = torch.from_numpy(s.G.data.copy()).cuda()
                f = lambda: mb.mapl_stiefel_step(U, G, 1e-2, retr, 5, None, ws)
                f()
                stream.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=stream):
                    f()
                g.replay()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for _ in range(reps):
                    g.replay()
                e1.record(stream)
                stream.synchronize()
                us = 1e3 * e0.elapsed_time(e1) / reps
                Uh = U.double()
                res = float(max(torch.linalg.matrix_norm(Uh[b].T @ Uh[b] - torch.eye(r, device="cuda", dtype=torch.float64))
                                for b in range(s.batch)))
                out[f"r{r}_{tag}"] = {"us_per_step": round(us, 1), "projector_steps_per_s": round(s.batch * 1e6 / us),
                                      "orth_residual_after": float(f"{res:.2e}")}
                if track_steps:
                    out[f"r{r}_{tag}"]["track"] = _stiefel_track(torch, mb, s, r, retr, ws, stream, track_steps)
    # full SPEL update (Eq. 4-7: tangent projection, momentum 0.95, 5 + 7 Newton-Schulz iterations), SURVEY 8f next row 2
    with torch.cuda.stream(stream):
        for r in (64, 128, 256, 512):
            s = I.make_stiefel(r)
            ws = mb.alloc_workspace(mb.mapl_spel_workspace_bytes(s.d, r, s.batch))
            U = torch.from_numpy(s.U.data.copy()).cuda()
            G = torch.from_numpy(s.G.data.copy()).cuda()
            Mom = torch.zeros_like(U)
            f = lambda: mb.mapl_spel_step(U, G, Mom, 2e-3, 0.95, 5, 7, ws)
            f()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                f()
            g.replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                g.replay()
            e1.record(stream)
            stream.synchronize()
            us = 1e3 * e0.elapsed_time(e1) / reps
            Uh = U.double()
            res = float(max(torch.linalg.matrix_norm(Uh[b].T @ Uh[b] - torch.eye(r, device="cuda", dtype=torch.float64))
                            for b in range(s.batch)))
            out[f"r{r}_spel"] = {"us_per_step": round(us, 1), "projector_steps_per_s": round(s.batch * 1e6 / us),
                                 "orth_residual_after": float(f"{res:.2e}")}
    out["config"] = ("d=2048, 3 projectors per call, fixed G, lr=1e-2, fp32; track: 1000 consecutive steps per variant, "
                     "residual in fp64 at the listed steps and max over all steps of the library's own per-step check "
                     "(info_out: an fp32 Gram of U, whose rounding floor is ~2e-8 r -- it reads high at r = 512)")
    return out


def centering_times(torch, mb, b, cfg, stream, reps=10):
    """SURVEY 8f next row 1 (Eq. 1 in full), measured beside the hot path on boundary 0 of the workload:
    mapl_center_table (once per parameter update), mapl_encode_centered (per micro-batch; compare calls_us.mapl_encode)
    and mapl_center_backward.  The sender's anchor factors are the boundary's A, B.  Graph-timed, us per call."""
    T = torch.empty((cfg.vocab, cfg.r), dtype=torch.float32, device="cuda")
    cws = mb.alloc_workspace(mb.mapl_center_workspace_bytes(b.desc))
    bws = mb.alloc_workspace(mb.mapl_center_backward_workspace_bytes(b.desc))
    dA = torch.empty_like(b.A)
    dU = torch.zeros_like(b.dU)
    fns = {
        "mapl_center_table": lambda: mb.mapl_center_table(b.desc, b.A, b.B, b.U, T, cws),
        "mapl_encode_centered": lambda: mb.mapl_encode_centered(b.desc, b.H, b.tok, T, b.U, b.C, b.Zq, b.codes, b.ws),
        "mapl_center_backward": lambda: mb.mapl_center_backward(b.desc, b.gz, b.tok, b.A, b.B, b.U, dA, None, dU, False, bws),
    }
    out = {}
    with torch.cuda.stream(stream):
        for name, f in fns.items():
            f()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                f()
            g.replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                g.replay()
            e1.record(stream)
            stream.synchronize()
            out[name] = round(1e3 * e0.elapsed_time(e1) / reps, 2)
    # grouped MCVQ (G=2, K=256, R=2) of the workload's [N,r] payload (gz of boundary 0)
    gen = torch.Generator(device="cuda").manual_seed(3)
    Cb = torch.randn((2, 256, cfg.r), device="cuda", generator=gen) * torch.tensor([1.0, 0.4], device="cuda")[:, None, None]
    codes8 = torch.empty((cfg.n_tokens, 2, cfg.r // 2), dtype=torch.uint8, device="cuda")
    Xq = torch.empty_like(b.gz)
    fns2 = {
        "mapl_mcvq_quantize": lambda: mb.mapl_mcvq_quantize(b.gz, Cb, codes8, None),
        "mapl_mcvq_dequantize": lambda: mb.mapl_mcvq_dequantize(codes8, Cb, Xq),
    }
    with torch.cuda.stream(stream):
        for name, f in fns2.items():
            f()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                f()
            g.replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                g.replay()
            e1.record(stream)
            stream.synchronize()
            out[name] = round(1e3 * e0.elapsed_time(e1) / reps, 2)
    out["mcvq_bytes_per_token"] = cfg.r  # (r/2) groups x 2 rounds x 1 byte
    # retained-energy diagnostic (Fig. 4b) and one micro-batch's codebook delta (a fifth of 2 x 256 rows)
    sums = torch.zeros(2, dtype=torch.float64, device="cuda")
    Zp = b.Zq if b.Zq is not None else b.gz
    idx = torch.arange(0, 512, 5, dtype=torch.int32, device="cuda")
    rows = torch.empty((idx.numel(), cfg.r), dtype=torch.float32, device="cuda")
    fns3 = {
        "mapl_energy_retained": lambda: mb.mapl_energy_retained(b.H, Zp, sums),
        "mapl_codebook_delta_pack+apply": lambda: (mb.mapl_codebook_delta_pack(Cb, idx, rows), mb.mapl_codebook_delta_apply(Cb, idx, rows)),
    }
    with torch.cuda.stream(stream):
        for name, f in fns3.items():
            f()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                f()
            g.replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                g.replay()
            e1.record(stream)
            stream.synchronize()
            out[name] = round(1e3 * e0.elapsed_time(e1) / reps, 2)
    out["note"] = "us per call, boundary 0; not part of the codec metric"
    return out


def roofline_step(cfg, peaks, ms_per_step, nb, calls_us):
    """Whole-config roofline: t_roof = sum over the three calls of max(bytes/peak_HBM, flops/peak_bf16),
    per boundary; `frac` compares it with the graph-timed codec time of a boundary (Stiefel step excluded)."""
    ab, af = alg_bytes_per_token(cfg), alg_flops_per_token(cfg)
    N = cfg.n_tokens
    t = {}
    for call in ("encode", "decode", "backward"):
        t[call] = 1e6 * max(ab[call] * N / (peaks["hbm"] * 1e9), af[call] * N / (peaks["bf16"] * 1e12))
    codec_us = sum(calls_us[k] for k in ("mapl_encode", "mapl_decode", "mapl_codec_backward"))
    # the same sum against the vendor's nominal peaks (8 TB/s HBM3e, 2.25 PFLOP/s dense bf16): context, SURVEY 8(d)
    t_nom = sum(1e6 * max(ab[c] * N / 8000e9, af[c] * N / 2250e12) for c in ("encode", "decode", "backward"))
    return {"t_roof_us_per_boundary": round(sum(t.values()), 2), "per_call_us": {k: round(v, 2) for k, v in t.items()},
            "measured_us_per_boundary": round(codec_us, 2), "frac": round(sum(t.values()) / codec_us, 3),
            "peaks": {"hbm_gbs": peaks["hbm"], "bf16_tflops": peaks["bf16"], "source": peaks["src"]},
            "nominal": {"t_roof_us_per_boundary": round(t_nom, 2), "frac": round(t_nom / codec_us, 3),
                        "hbm_gbs": 8000, "bf16_tflops": 2250}}


def roofline_for(name, k, cfg, peaks, total_ms):
    """achieved = algorithmic bytes (or flops) of one launch / its measured average duration."""
    N = cfg.n_tokens
    ab, af = alg_bytes_per_token(cfg), alg_flops_per_token(cfg)
    avg_s = 1e-3 * k["ms"] / k["launches"]
    # which call the kernel belongs to and the share of that call's algorithmic work it carries
    call = {"k_tc_encode": "encode", "k_tc_encode_rvq": "encode", "k_simt_encode_rvq": "encode",
            "k_tc_decode": "decode", "k_tc_bwd_gz": "backward", "k_tc_bwd_du": "backward"}.get(name)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        for line in open(tpath).read().splitlines()[1:]:
            wl, kern_name, nbytes = line.split(",")
            if wl == cfg.name and kern_name == name:
                traffic = int(nbytes)
    if call is None:
        return {"kernel": name, "bound": "hbm", "achieved": None, "peak": peaks["hbm"], "unit": "GB/s", "frac": None,
                "traffic": traffic, "note": "generic kernel shared by several calls; see kernels"}
    byt, flo = ab[call] * N, af[call] * N
    if name == "k_tc_bwd_gz":     # reads g, tok, writes gz, dH  (H and payload are read by k_tc_bwd_du)
        s = 2 if cfg.act_dtype == "bf16" else 4
        byt = (2 * cfg.d * s + cfg.r * s + 4) * N
        flo = (4 * cfg.d * cfg.r + 2 * cfg.d * cfg.anchor_rank) * N
    if name == "k_tc_bwd_du":
        s = 2 if cfg.act_dtype == "bf16" else 4
        byt = (2 * cfg.d * s + 2 * cfg.r * s) * N
        flo = 4 * cfg.d * cfg.r * N
    t_hbm, t_tc = byt / (peaks["hbm"] * 1e9), flo / (peaks["bf16"] * 1e12)
    if t_hbm >= t_tc:
        ach = byt / avg_s / 1e9
        return {"kernel": name, "bound": "hbm", "achieved": ach, "peak": peaks["hbm"], "unit": "GB/s",
                "frac": ach / peaks["hbm"], "traffic": traffic, "peak_source": peaks["src"] + " (burst copy)",
                "avg_us": avg_s * 1e6, "alg_bytes_per_launch": byt,
                "note": "avg_us is event-bracketed per launch (no dependent-launch overlap, ~5 us of launch latency "
                        "inside the pair): a lower bound on frac; calls_us / roofline_step are graph-timed"}
    ach = flo / avg_s / 1e12
    return {"kernel": name, "bound": "tensor", "achieved": ach, "peak": peaks["bf16"], "unit": "TFLOP/s",
            "frac": ach / peaks["bf16"], "traffic": traffic, "peak_source": peaks["src"] + " (burst bf16)",
            "avg_us": avg_s * 1e6, "alg_flops_per_launch": flo,
            "note": "avg_us is event-bracketed per launch (no dependent-launch overlap): a lower bound on frac; "
                    "calls_us / roofline_step are graph-timed"}


# ---------------------------------------------------------------- the oracle arm (CPU baseline)

def _oracle_pass(cfg, n, boundary):
    """One enc + dec + full bwd of `n` contiguous tokens of one boundary through the fp64 oracle."""
    from oracle import mapl_oracle as o
    from paper_2606_05484_b200 import inputs as I
    bi = I.make_boundary(cfg.with_tokens(n), boundary)
    H, U, g = bi.H.f64, bi.U.f64, bi.g.f64
    t0 = time.perf_counter()
    enc = o.encode(H, U, bi.C.f64 if bi.C is not None else None)
    Hhat = o.decode(enc["Zhat"], U, bi.tok, bi.A.f64, bi.B.f64)
    bw = o.backward(g, H, enc["Zhat"], U, bi.tok, bi.A.f64, bi.B.f64, want_dB=False)
    dt = time.perf_counter() - t0
    del Hhat, bw
    return dt


def cpu_baseline(cfg, budget_s=20.0, sample_tokens=None):
    """The fp64 oracle, as it stands, on the host cores: contiguous token samples of the workload's
    boundaries, sized and repeated until about budget_s / 2 seconds of oracle work have been timed."""
    from oracle import mapl_oracle as o
    if sample_tokens:
        dt = _oracle_pass(cfg, sample_tokens, 0)
        return {"value": sample_tokens / dt, "unit": UNIT, "cores": o.threads(), "kind": "oracle",
                "sample": f"{sample_tokens} contiguous tokens of boundary 0 (enc+dec+bwd, fp64), {dt:.1f} s"}
    n = min(cfg.n_tokens, 512)
    dt = _oracle_pass(cfg, n, 0)                                   # sizing probe, not counted
    n = int(min(cfg.n_tokens, max(n, n * (budget_s / 4) / max(dt, 1e-3))))
    t_used, tokens, passes = 0.0, 0, 0
    while t_used < budget_s / 2 and passes < 64:
        t_used += _oracle_pass(cfg, n, passes % max(1, cfg.n_boundaries))
        tokens += n
        passes += 1
    return {"value": tokens / t_used, "unit": UNIT, "cores": o.threads(), "kind": "oracle",
            "sample": f"{passes} passes of {n} contiguous tokens over the workload's boundaries (enc+dec+bwd, fp64), "
                      f"{t_used:.1f} s of oracle time"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores.  Each of the K steps is a
    bounded contiguous-token sample of the workload, sized from one untimed probe so that the whole
    run ends within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, wdesc = workload(args.workload)
    probe_n = 256
    probe = cpu_baseline(cfg, sample_tokens=probe_n)
    rate = probe["value"]
    n = int(max(64, min(cfg.n_tokens, rate * 90.0 / max(1, args.steps + args.warmup))))
    for _ in range(args.warmup):
        cpu_baseline(cfg, sample_tokens=n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        last = cpu_baseline(cfg, sample_tokens=n)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    cb = {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle",
          "sample": f"{n} contiguous tokens of boundary 0 per step (enc+dec+bwd, fp64), {args.steps} steps"}
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": wdesc}, "cpu_baseline": cb,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="mapl", choices=["mapl", "reference"])
    ap.add_argument("--workload", default="c1", choices=["c1", "c2", "c3", "c0"])
    ap.add_argument("--tokens", type=int, default=0, help="override tokens per boundary (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stiefel", action="store_true", help="skip the configs[4] Stiefel-step sweep")
    ap.add_argument("--track-steps", type=int, default=1000,
                    help="configs[4]: consecutive Stiefel steps per variant with the orthogonality residual tracked (0 = off)")
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mapl(args)


if __name__ == "__main__":
    main()
