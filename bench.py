#!/usr/bin/env python
"""bench.py -- decoded TPC clusters/s of the track-model decoder on synthetic time frames (BASELINE.json metric).

One "step" = one pass of the whole hot path over one synthetic time frame:
`tmd_decode(flags = 0)` through the C ABI, compressed SoA resident in HBM.  Prints ONE JSON line (see the task contract):
value = clusters decoded per second over all ranks (device-timed with CUDA events, max over ranks), `e2e` = the same
through `tmd_decode_host_async` with pinned HOST buffers (copies inside the timed region), `roofline` for the dominant
kernel (timed live, outside the timed region, with CUDA events the library records on the launching stream) with the
instruction-issue bound beside the HBM bound, `cpu_baseline` = the CPU oracle on a bounded sample of the same workload
(one core, and all host cores), `other_workloads` = the same step timed on c2, c4 and a batch of 64 c1 frames.

Multi-GPU: the path does not shard ("replicas only") -- every rank decodes its own time frame
(different seed), no collective on the data path; torch.distributed (NCCL) is used for the barrier and the max.
`python bench.py --gpus N` outside torchrun starts the N ranks itself (torch.distributed.run on 127.0.0.1).

`--impl reference` times the CPU oracle (oracle/, as it stands, single thread) on bounded samples of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

BZ = 0.5
METRIC = "decoded_tpc_clusters_per_second"
UNIT = "clusters/s"
BATCH_FRAMES = 64          # other_workloads["c1x64"]: SURVEY.md §8(f)-4, many small frames in one call


def algorithmic_bytes_attached(n_trk: int, n_att: int) -> int:
    """per-track 11 B + copy-through 7 B/cluster + residual streams 8 B/residual in, 16 B/cluster out."""
    return 11 * n_trk + 7 * n_att + 8 * (n_att - n_trk) + 16 * n_att


def algorithmic_bytes_unattached(n_un: int, n_bins: int) -> int:
    return 13 * n_un + 4 * n_bins + 16 * n_un + 4 * (n_bins + 1)


def kernel_algorithmic_bytes(n_trk: int, n_att: int, n_un: int, n_bins: int) -> dict:
    """The share of the algorithmic bytes each kernel is there to move: the decode kernel consumes the
    per-track fields and the four residual streams, the scatter kernel the copy-through fields and writes the records,
    the unattached kernel its 13 B in / 16 B out.  The rank and scan kernels move no algorithmic byte (overhead)."""
    return {"track_decode": 11 * n_trk + 8 * (n_att - n_trk), "scatter": 7 * n_att + 16 * n_att,
            "unattached": algorithmic_bytes_unattached(n_un, n_bins)}


# ------------------------------------------------------------------------------------------------ workload on the device
def build_workload(name: str, device, seed_offset: int = 0, keep_truth: bool = False, scale: float = 1.0):
    """Synthetic time frame `name` (tmd_inputs.timeframe.WORKLOADS) as device tensors of the compressed SoA: cluster truth
    (helix tracks + unattached clusters) -> the library's own encoder (tmd_encode_attached + tmd_encode_unattached), itself
    checked byte for byte against the oracle encoder in the -m gpu tests (bench.py may not run the oracle here)."""
    import torch
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs import build_geometry, timeframe as tf

    geo = build_geometry(36)
    mk, n_un, single = tf.WORKLOADS[name]
    cfg = mk()
    cfg.seed += 1000 * seed_offset
    if scale != 1.0:                                        # a fraction of the frame, same recipe (entropy-stage measurement)
        cfg.n_tracks, n_un = max(1, int(cfg.n_tracks * scale)), int(n_un * scale)
    truth = tf.generate_truth(cfg, geo, device, batch=2_000_000)
    n_trk, n_att = truth.n_tracks, truth.n_attached
    arrays = {"trk_ncl": truth.trk_ncl}
    spec = dict(T.COMPRESSED_ARRAYS)
    tdt = {"<u2": torch.int16, "i1": torch.int8, "u1": torch.uint8, "<u4": torch.int32}
    for k in ("trk_qpt", "trk_row0", "trk_sec0", "trk_pad0", "trk_time0"):
        arrays[k] = torch.empty(n_trk, dtype=tdt[spec[k]], device=device)
    for k in ("a_qtot", "a_qmax", "a_flags", "a_sigpad", "a_sigtime"):
        arrays[k] = torch.empty(n_att, dtype=tdt[spec[k]], device=device)
    for k in ("a_rowdiff", "a_secleg", "a_padres", "a_timeres"):
        arrays[k] = torch.empty(n_att - n_trk, dtype=tdt[spec[k]], device=device)
    ctx = T.tmd_create(geo, BZ)
    ws = torch.empty(T.tmd_workspace_bytes(ctx, n_trk, n_att, 0), dtype=torch.uint8, device=device)
    T.tmd_encode_attached(ctx, truth.trk_ncl, truth.trk_qptf, truth.att, truth.leg, arrays, ws,
                          torch.cuda.current_stream().cuda_stream)
    del ws
    un = tf.generate_unattached_truth(geo, n_un, cfg.seed, device, "inv_x", single)
    n_u = int(un.shape[0])
    for k in ("u_qtot", "u_qmax", "u_flags", "u_sigpad", "u_sigtime", "u_paddiff", "u_timediff"):
        arrays[k] = torch.empty(n_u, dtype=tdt[spec[k]], device=device)
    arrays["u_bin_count"] = torch.empty(geo.n_bins, dtype=torch.int32, device=device)
    ws = torch.empty(T.tmd_encode_unattached_workspace_bytes(ctx, n_u), dtype=torch.uint8, device=device)
    T.tmd_encode_unattached(ctx, un, arrays, ws, torch.cuda.current_stream().cuda_stream)
    T.tmd_destroy(ctx)
    del ws
    if keep_truth:
        truth.un = un
    else:
        truth = None
    del un
    torch.cuda.empty_cache()
    return (geo, arrays, truth) if keep_truth else (geo, arrays)


def oracle_sample(workload: str, n_s: int, device):
    """A bounded sample of `workload` for the CPU oracle: the first n_s tracks of the same generator recipe (same pT / length /
    looper mix) and the same fraction of the unattached clusters.  All of them are ENCODED BY THE ORACLE'S OWN ENCODER --
    nothing the oracle reads comes from the CUDA path."""
    from tmd_inputs import build_geometry, physical as ph, timeframe as tf
    from oracle import tmd_oracle as O

    geo = build_geometry(36)
    mk, n_un, single = tf.WORKLOADS[workload]
    cfg = mk()
    n_s = min(cfg.n_tracks, n_s)
    frac = n_s / cfg.n_tracks
    cfg.n_tracks = n_s
    tr = tf.generate_truth(cfg, geo, device, batch=400_000)
    ev_att = tr.att.cpu().numpy().view(ph.CLUSTER_DTYPE).reshape(-1)
    un = tf.generate_unattached_truth(geo, int(n_un * frac), cfg.seed, device, "inv_x", single)
    comp = O.encode(geo, BZ, tr.trk_ncl.cpu().numpy().view(np.uint16), tr.trk_qptf.cpu().numpy(), ev_att, tr.leg.cpu().numpy(),
                    un.cpu().numpy().view(ph.CLUSTER_DTYPE).reshape(-1))
    return geo, comp, n_s


def time_oracle(geo, comp) -> float:
    from oracle import tmd_oracle as O
    t0 = time.perf_counter()
    O.decode(geo, BZ, comp)
    return time.perf_counter() - t0


def host_description() -> dict:
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count()}


def oracle_all_cores(geo, comp, seconds: float = 4.0) -> dict | None:
    """The same oracle on ALL host cores: one process per core, each decoding the same bounded sample repeatedly for about
    `seconds` ("one B200 = N_eq host cores").  Independent processes = independent time frames, which is
    how the path scales on a CPU farm (PAPER.md L70 compares one GPU with N EPN cores)."""
    import tempfile
    from tmd_inputs.layout import COMPRESSED_FIELDS
    n_proc = os.cpu_count() or 1
    one = time_oracle(geo, comp)
    reps = max(1, int(seconds / max(one, 1e-3)))
    with tempfile.TemporaryDirectory(dir="/dev/shm" if os.path.isdir("/dev/shm") else None) as d:
        np.savez(os.path.join(d, "sample.npz"), **{k: getattr(comp, k) for k in COMPRESSED_FIELDS})
        cmd = [sys.executable, os.path.abspath(__file__), "--oracle-worker", os.path.join(d, "sample.npz"), "--oracle-reps", str(reps)]
        procs = [subprocess.Popen(cmd, stdout=subprocess.PIPE, text=True) for _ in range(n_proc)]
        spans = []
        for p in procs:
            out, _ = p.communicate(timeout=600)
            if p.returncode != 0:
                return None
            t0, t1 = (float(v) for v in out.strip().split()[-2:])
            spans.append((t0, t1))
    wall = max(t1 for _, t1 in spans) - min(t0 for t0, _ in spans)      # time.time() stamps: first start to last end
    n_cl = comp.n_attached + comp.n_unattached
    return {"processes": n_proc, "value": n_proc * reps * n_cl / wall, "unit": UNIT, "reps_per_process": reps}


def oracle_worker(path: str, reps: int) -> None:
    from tmd_inputs import build_geometry
    from tmd_inputs.layout import Compressed
    z = np.load(path)
    comp = Compressed(**{k: z[k] for k in z.files})
    geo = build_geometry(36)
    time_oracle(geo, comp)                       # builds / loads liborc.so, touches the pages
    t0 = time.time()
    for _ in range(reps):
        time_oracle(geo, comp)
    print(t0, time.time())


def cpu_baseline(workload: str, n_s: int, device, gpu_value: float, all_cores: bool) -> dict:
    """The oracle as it stands (single thread) timed on a bounded sample of the workload (about 10 s of decoding at c3)."""
    geo, comp, n_s = oracle_sample(workload, n_s, device)
    dt = time_oracle(geo, comp)
    n_cl = comp.n_attached + comp.n_unattached
    out = {"value": n_cl / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"{n_s} tracks of the {workload} recipe ({comp.n_attached} attached) + the same fraction of the unattached "
                     f"clusters ({comp.n_unattached}), encoded by the oracle encoder; oracle/tmd_oracle.c orc_decode, single "
                     f"thread, {dt:.2f} s",
           "host": host_description(), "gpu_equals_host_cores": gpu_value / (n_cl / dt)}
    if all_cores:
        small = oracle_sample(workload, max(1000, n_s // 100), device)
        out["all_cores"] = oracle_all_cores(small[0], small[1])
    return out


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """SM clock, power and throttle reasons sampled through NVML every few milliseconds DURING the timed region."""
    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, gpu_index: int, period_s: float = 0.004):
        import threading
        self.samples, self.err, self.stop_flag, self.period = [], None, False, period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[gpu_index]) if vis and vis.split(",")[gpu_index].isdigit() else gpu_index
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # noqa: BLE001 -- no NVML: report it in the JSON line
            self.err = f"nvml unavailable: {e}"
            return
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()

    def _run(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                self.samples.append((float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)),
                                     nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0,
                                     int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))))
            except Exception as e:  # noqa: BLE001
                self.err = f"nvml sample failed: {e}"
                return
            time.sleep(self.period)

    def stop(self) -> dict:
        if self.err and not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [self.err]}
        self.stop_flag = True
        self.th.join()
        sm = [x[0] for x in self.samples]
        power = [x[1] for x in self.samples]
        mask = 0
        for x in self.samples:
            mask |= x[2]
        reasons = sorted(k for k, b in {**self.BAD, **self.NOTE}.items() if mask & b)
        thr = 0.5 * (min(power) + max(power))          # "under load" = samples in the upper half of the power range seen
        load = [c for c, p in zip(sm, power) if p >= thr] or sm
        return {"sm_mhz": float(np.median(load)), "sm_max_mhz": self.sm_max, "reasons": reasons, "samples": len(sm),
                "power_w_max": max(power)}


# ------------------------------------------------------------------------------------------------ ranks
def aggregate_over_ranks(total_ms: float, n_units: float, device):
    """Replicas only: every rank decodes its own time frame.  The job's time is the MAX over ranks of the
    device time, its work the SUM of the units; no collective on the data path.  Works on any backend (NCCL on GPUs,
    gloo in the CPU test)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return total_ms, n_units
    t = torch.tensor([total_ms, n_units], dtype=torch.float64, device=device)
    tmax = t.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    tsum = t.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(tsum[1])


def rank_seed_offset(rank: int) -> int:
    """Rank r decodes time frame r of the recipe (seed + 1000 r): different data, same size class (weak scaling)."""
    return rank


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(n: int, argv: list[str]) -> int:
    """`python bench.py --gpus N` outside torchrun: start the N ranks (one per GPU) the way the driver does."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(free_port()), os.path.abspath(__file__), *argv]
    return subprocess.call(cmd)


def run_rank_logic_only(args) -> None:
    """The multi-rank plumbing of run_ours without a GPU (gloo): which frame a rank takes, max of times, sum of clusters.
    Used by tests/test_multi_rank.py through `bench.py --gpus 2 --rank-logic-only`."""
    import torch
    import torch.distributed as dist
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    ms, n = aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 + rank_seed_offset(rank), torch.device("cpu"))
    if rank == 0:
        print(json.dumps({"metric": METRIC, "n_gpus": world, "ms_per_step": ms, "value": n / (ms * 1e-3), "unit": UNIT,
                          "scaling": "weak", "rank_logic_only": True}), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------ timing helpers
class Frame:
    """One time frame resident in HBM with its outputs and workspace."""

    def __init__(self, T, ctx, geo, arrays, device):
        import torch
        self.arrays = arrays
        self.n_trk, self.n_att, self.n_un = (int(arrays[k].shape[0]) for k in ("trk_ncl", "a_qtot", "u_qtot"))
        self.n_cl, self.n_bins = self.n_att + self.n_un, geo.n_bins
        self.clusters = torch.empty(max(self.n_cl, 1) * 16, dtype=torch.uint8, device=device)
        self.bin_offset = torch.empty(geo.n_bins + 1, dtype=torch.int32, device=device)
        self.ws = torch.empty(T.tmd_workspace_bytes(ctx, self.n_trk, self.n_att, self.n_un), dtype=torch.uint8, device=device)
        self.comp = T.make_compressed(arrays)
        self.out = T.make_output(self.clusters, self.bin_offset, self.ws)

    def algorithmic_bytes(self) -> int:
        return algorithmic_bytes_attached(self.n_trk, self.n_att) + algorithmic_bytes_unattached(self.n_un, self.n_bins)


def timed_steps(step, steps: int, warmup: int, barrier) -> list[float]:
    """W untimed calls of `step`, then K timed ones, one CUDA-event pair per step on torch's current stream (the stream the
    library launches on), bracketed by barrier + synchronize on both sides.  Returns the K per-step times in ms."""
    import torch
    for _ in range(warmup):
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for s0, s1 in ev:
        s0.record()
        step()
        s1.record()
    barrier()
    return [a.elapsed_time(b) for a, b in ev]


def per_kernel_ms(T, ctx, frame: Frame, stream, n: int = 3) -> dict:
    """OUTSIDE the timed region: the same step with an event pair around every kernel (TMD_TIMING), averaged over n runs."""
    import torch
    acc: dict[str, float] = {}
    for _ in range(n):
        T.tmd_decode(ctx, frame.comp, frame.out, T.TMD_TIMING, stream)
        for name, ms in T.tmd_kernel_times(ctx):
            acc[name] = acc.get(name, 0.0) + ms / n
    torch.cuda.synchronize()
    return acc


def stats(ms: list[float]) -> dict:
    return {"mean": float(np.mean(ms)), "median": float(np.median(ms)), "min": float(np.min(ms))}


def side_workload(T, name: str, device, steps: int, peak: float) -> dict:
    """ms/step, clusters/s and path fraction of another BASELINE.json config, measured like the main one (single rank)."""
    import torch
    geo, arrays = build_workload(name, device)
    ctx = T.tmd_create(geo, BZ)
    fr = Frame(T, ctx, geo, arrays, device)
    stream = torch.cuda.current_stream().cuda_stream
    ms = timed_steps(lambda: T.tmd_decode(ctx, fr.comp, fr.out, 0, stream), steps, 3, torch.cuda.synchronize)
    kms = per_kernel_ms(T, ctx, fr, stream)
    T.tmd_destroy(ctx)
    st = stats(ms)
    gbs = fr.algorithmic_bytes() / (st["mean"] * 1e-3) / 1e9
    return {"n_tracks": fr.n_trk, "n_attached": fr.n_att, "n_unattached": fr.n_un, "steps": steps, "ms_per_step": st["mean"],
            "ms_per_step_median": st["median"], "ms_per_step_min": st["min"], "value": fr.n_cl / (st["mean"] * 1e-3), "unit": UNIT,
            "path_gbs": gbs, "path_frac_of_hbm_peak": gbs / peak, "kernel_ms": kms,
            "l2": "inputs larger than L2, no flush" if fr.algorithmic_bytes() > 400e6 else "L2-resident workload (flag)"}


def two_in_flight(T, ctx, geo, arrays, device, steps: int, one_frame_ms: float) -> dict:
    """"multiple instances are executed concurrently on different streams".  Two time frames (the same
    compressed arrays, read-only; outputs and workspace of their own) decoded by two plain tmd_decode calls per step on two
    streams, so that one frame's memory-bound kernels can run beside the other's issue-bound track decode.  Measured twice:
    both streams at the default priority, and the second stream at high priority.  value = clusters of both frames over the
    time from the common start to the later of the two ends (CUDA events)."""
    import torch
    frames = [Frame(T, ctx, geo, arrays, device) for _ in range(2)]
    out = {"frames_in_flight": 2, "steps": steps, "one_frame_at_a_time_ms": one_frame_ms}
    cur = torch.cuda.current_stream()
    for label, prio in (("equal_priority", 0), ("second_stream_high_priority", -1)):
        streams = [torch.cuda.Stream(device=device, priority=0), torch.cuda.Stream(device=device, priority=prio)]

        def run(k: int) -> float:
            torch.cuda.synchronize()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record(cur)
            for st, fr in zip(streams, frames):
                st.wait_event(t0)
                for _ in range(k):
                    T.tmd_decode(ctx, fr.comp, fr.out, 0, st.cuda_stream)
                cur.wait_stream(st)
            t1.record(cur)
            torch.cuda.synchronize()
            return t0.elapsed_time(t1)
        run(3)
        ms = run(steps) / steps                               # per pair of frames
        out[label] = {"ms_per_two_frames": ms, "value": 2 * frames[0].n_cl / (ms * 1e-3), "unit": UNIT,
                      "speedup_vs_one_at_a_time": 2 * one_frame_ms / ms}
    del frames
    torch.cuda.empty_cache()
    return out


def batch_workload(T, device, n_frames: int, steps: int, peak: float) -> dict | None:
    """n_frames c1-sized frames (single Pb-Pb-like events, different seeds) decoded by ONE
    tmd_decode_batch call, next to the same frames decoded one tmd_decode call after the other."""
    import torch
    if not hasattr(T, "tmd_decode_batch"):
        return None
    frames, geo = [], None
    ctx = None
    for i in range(n_frames):
        geo, arrays = build_workload("c1", device, seed_offset=i)
        if ctx is None:
            ctx = T.tmd_create(geo, BZ)
        frames.append(Frame(T, ctx, geo, arrays, device))
    stream = torch.cuda.current_stream().cuda_stream
    comps, outs = [f.comp for f in frames], [f.out for f in frames]
    batch = T.make_batch(comps, outs)
    ms_b = timed_steps(lambda: T.tmd_decode_batch(ctx, batch, 0, stream), steps, 3, torch.cuda.synchronize)

    def one_by_one():
        for c, o in zip(comps, outs):
            T.tmd_decode(ctx, c, o, 0, stream)
    ms_s = timed_steps(one_by_one, steps, 3, torch.cuda.synchronize)
    ms_1 = timed_steps(lambda: T.tmd_decode(ctx, comps[0], outs[0], 0, stream), steps, 3, torch.cuda.synchronize)
    T.tmd_decode_batch(ctx, batch, T.TMD_TIMING, stream)
    kms: dict[str, float] = {}
    for name, ms in T.tmd_kernel_times(ctx):
        kms[name] = kms.get(name, 0.0) + ms
    T.tmd_destroy(ctx)
    n_cl = sum(f.n_cl for f in frames)
    alg = sum(f.algorithmic_bytes() for f in frames)
    sb, ss, s1 = stats(ms_b), stats(ms_s), stats(ms_1)
    return {"frames": n_frames, "clusters": n_cl, "steps": steps, "ms_per_step": sb["mean"], "ms_per_step_median": sb["median"],
            "ms_per_step_min": sb["min"], "value": n_cl / (sb["mean"] * 1e-3), "unit": UNIT,
            "path_gbs": alg / (sb["mean"] * 1e-3) / 1e9, "path_frac_of_hbm_peak": alg / (sb["mean"] * 1e-3) / 1e9 / peak,
            "same_frames_one_call_each": {"ms": ss["mean"], "value": n_cl / (ss["mean"] * 1e-3)},
            "single_c1_frame": {"ms": s1["mean"], "value": frames[0].n_cl / (s1["mean"] * 1e-3)}, "kernel_ms": kms,
            "l2": "each frame is L2-sized; 64 frames = 3 GB of traffic per step, no flush"}


def entropy_workload(T, device, steps: int, peak: float, workload: str) -> dict | None:
    """the entropy stage in front (PAPER.md L49 'TPC Entropy Decoding').  The WHOLE frame of `workload`
    (c3: 4.8 GB of arrays, a ~2.1 GB container) is written as a TMDZ container by the library's HOST encoder (one core,
    outside any timed region, ~20 s at c3), copied to the device, and the GPU rANS decode into the compressed SoA is timed
    alone and chained with tmd_decode on the same stream."""
    import torch
    if not hasattr(T, "tmd_entropy_decode"):
        return None
    geo, arrays = build_workload(workload, device)
    host = {k: v.cpu() for k, v in arrays.items()}
    t0 = time.perf_counter()
    blob = T.tmd_entropy_encode_host(host, geo.n_bins)
    enc_s = time.perf_counter() - t0
    raw = sum(v.numel() * v.element_size() for v in arrays.values())
    d_blob = torch.from_numpy(blob).to(device)
    d_err = torch.zeros(1, dtype=torch.int32, device=device)
    out = {k: torch.empty_like(v) for k, v in arrays.items()}
    head = blob[:T.ENTROPY_HEAD_BYTES]
    stream = torch.cuda.current_stream().cuda_stream
    ms_z = timed_steps(lambda: T.tmd_entropy_decode(head, d_blob, out, d_err, stream), steps, 3, torch.cuda.synchronize)
    same = all(torch.equal(out[k], arrays[k]) for k in arrays) and int(d_err.item()) == 0
    ctx = T.tmd_create(geo, BZ)
    fr = Frame(T, ctx, geo, out, device)

    def chain():
        T.tmd_entropy_decode(head, d_blob, out, d_err, stream)
        T.tmd_decode(ctx, fr.comp, fr.out, 0, stream)
    ms_c = timed_steps(chain, steps, 3, torch.cuda.synchronize)
    sz, sc = stats(ms_z), stats(ms_c)
    n_att_, n_un_, n_cl_ = fr.n_att, fr.n_un, fr.n_cl
    # ---- container in, clusters out, host to host (tmd_decode_container_host_async): the e2e leg again, with the 2.3x smaller
    #      container on the bus instead of the arrays; same two-slot pipeline, same wall-clock timing, copies inside
    del fr, out, arrays, d_blob
    torch.cuda.empty_cache()
    h_blob = torch.from_numpy(blob).pin_memory()
    keep, houts = [], []
    for _ in range(T.TMD_HOST_SLOTS):
        hc = torch.empty(n_cl_ * 16, dtype=torch.uint8, pin_memory=True)
        hb = torch.empty(geo.n_bins + 1, dtype=torch.int32, pin_memory=True)
        keep.append((hc, hb)); houts.append(T.make_output(hc, hb))
    for s_ in range(T.TMD_HOST_SLOTS):
        T.tmd_decode_container_host_async(ctx, h_blob, houts[s_], 0, s_)
    for s_ in range(T.TMD_HOST_SLOTS):
        T.tmd_host_wait(ctx, s_)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(steps):
        T.tmd_decode_container_host_async(ctx, h_blob, houts[i % T.TMD_HOST_SLOTS], 0, i % T.TMD_HOST_SLOTS)
    for s_ in range(T.TMD_HOST_SLOTS):
        T.tmd_host_wait(ctx, s_)
    pipe_s = time.perf_counter() - t0
    t0 = time.perf_counter()
    T.tmd_decode_container_host_async(ctx, h_blob, houts[0], 0, 0)
    T.tmd_host_wait(ctx, 0)
    single_s = time.perf_counter() - t0
    e2e_container = {"value": n_cl_ * steps / pipe_s, "unit": UNIT, "h2d_bytes_per_step": int(h_blob.numel()),
                     "d2h_bytes_per_step": int(keep[0][0].numel() + keep[0][1].numel() * 4), "steps": steps,
                     "mode": "two-slot pipeline, tmd_decode_container_host_async (upload container, entropy decode, decode, download)",
                     "single_frame_ms": 1e3 * single_s}
    T.tmd_destroy(ctx)
    del keep, houts, h_blob
    return {"workload": f"full {workload} frame", "e2e_container": e2e_container, "n_attached": n_att_, "n_unattached": n_un_, "raw_bytes": raw, "container_bytes": int(blob.size),
            "compression": raw / blob.size, "restores_the_arrays": bool(same), "entropy_decode_ms": sz["mean"], "entropy_decode_ms_min": sz["min"],
            "entropy_decode_out_gbs": raw / (sz["mean"] * 1e-3) / 1e9, "entropy_decode_frac_of_hbm_peak": (raw + blob.size) / (sz["mean"] * 1e-3) / 1e9 / peak,
            "chain_ms": sc["mean"], "chain_clusters_per_s": n_cl_ / (sc["mean"] * 1e-3), "host_encode_s": enc_s,
            "l2": "container (%.0f MB) + arrays (%.0f MB): %s" % (blob.size / 1e6, raw / 1e6, "larger than L2, no flush"
                                                                  if blob.size + raw > 400e6 else "partly L2-resident (flag)")}


KERNEL_SOURCES = ("tmd_api.cu", "tmd_common.cuh", "tmd_decode.cuh", "tmd_rank.cuh", "tmd_scan.cuh", "tmd_scatter.cuh", "tmd_sort.cuh",
                  "tmd_unattached.cuh")


def kernel_source_hash() -> str:
    """sha256 (first 12 hex digits) over the sources of the kernels of one tmd_decode step and their launch code: the key that
    ties profiles/traffic.txt (numbers read from an ncu capture) to the tree they were captured from."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        h.update(open(os.path.join(ROOT, "paper_2411_02206_b200", "csrc", name), "rb").read())
    return h.hexdigest()[:12]


def ncu_profile_numbers(kernel: str, workload: str):
    """(dram bytes per launch, warp instructions per launch, observed bound, source) of `kernel` from the committed ncu summary
    profiles/traffic.txt (`workload kernel dram_bytes warp_inst observed-bound...`; a line `sources <hash>` names the kernel
    sources the capture was made from).  If the kernels changed since (hash differs), the numbers are REFUSED: (None, None,
    None, reason)."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    found, captured = None, None
    try:
        for line in open(path):
            v = line.split()
            if len(v) >= 2 and v[0] == "sources":
                captured = v[1]
            if len(v) >= 3 and v[0] == workload and v[1] == kernel:
                found = (float(v[2]), float(v[3]) if len(v) >= 4 else None, " ".join(v[4:]) or None)
    except OSError:
        return None, None, None, None
    if found is None:
        return None, None, None, None
    now = kernel_source_hash()
    if captured != now:
        return None, None, None, f"stale: profiles/traffic.txt was captured from kernel sources {captured}, the tree is {now}"
    return (*found, f"profiles/traffic.txt (kernel sources {now})")


# ------------------------------------------------------------------------------------------------ arms
def run_ours(args) -> None:
    import torch
    import torch.distributed as dist
    from paper_2411_02206_b200 import tmd as T

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)

    geo, arrays = build_workload(args.workload, device, seed_offset=rank_seed_offset(rank))
    ctx = T.tmd_create(geo, BZ)
    fr = Frame(T, ctx, geo, arrays, device)
    n_trk, n_att, n_un, n_cl = fr.n_trk, fr.n_att, fr.n_un, fr.n_cl
    stream = torch.cuda.current_stream().cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- the timed region: K production calls (flags = 0), nothing else
    for _ in range(args.warmup):
        T.tmd_decode(ctx, fr.comp, fr.out, 0, stream)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    step_ms = timed_steps(lambda: T.tmd_decode(ctx, fr.comp, fr.out, 0, stream), args.steps, 0, barrier)
    clocks = sampler.stop() if sampler else None
    launches = T.tmd_last_launch_count(ctx) * args.steps
    total_ms, n_cl_all = aggregate_over_ranks(sum(step_ms), float(n_cl), device)
    ms_per_step = total_ms / args.steps
    value = n_cl_all / (ms_per_step * 1e-3)
    # ---- outside the timed region: per-kernel times (event pair around every kernel) for the roofline of the dominant kernel
    kms = per_kernel_ms(T, ctx, fr, stream)
    overlap = None
    if world == 1 and rank == 0 and not args.no_extras:
        overlap = two_in_flight(T, ctx, geo, arrays, device, min(args.steps, 10), sum(step_ms) / args.steps)

    # ---- end to end: pinned host buffers in, pinned host buffers out, every copy inside the timed region.  Frames go
    #      through the library's two-slot pipeline (tmd_decode_host_async): the upload of frame i+1 runs beside the
    #      download of frame i, as in the paper's deployment; each slot has its own output buffers.
    h_in = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in arrays.items()}
    h2d = sum(v.numel() * v.element_size() for v in h_in.values())
    alg_total = fr.algorithmic_bytes()
    del fr, arrays
    torch.cuda.empty_cache()
    hcomp = T.make_compressed(h_in)
    houts, keep = [], []
    # One rank alone pins an output buffer per pipeline slot (download of frame i beside upload of frame i+1).  With several
    # ranks on one host that is 15 GB of page-locked memory per rank (123 GB at 8 ranks): they pin ONE output buffer and use
    # one slot, i.e. upload, decode and download of a rank's frames run one after the other (the line says so in e2e.mode).
    e2e_slots = T.TMD_HOST_SLOTS if world == 1 else 1
    for _ in range(e2e_slots):
        hc = torch.empty(n_cl * 16, dtype=torch.uint8, pin_memory=True)
        hb = torch.empty(geo.n_bins + 1, dtype=torch.int32, pin_memory=True)
        keep.append((hc, hb))
        houts.append(T.make_output(hc, hb))
    d2h = keep[0][0].numel() + keep[0][1].numel() * 4
    e2e_steps = max(2, min(args.steps, args.e2e_steps))
    for s_ in range(e2e_slots):                               # warm-up: allocates the slots' device arenas
        T.tmd_decode_host_async(ctx, hcomp, houts[s_], 0, s_)
    for s_ in range(e2e_slots):
        T.tmd_host_wait(ctx, s_)
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        T.tmd_decode_host_async(ctx, hcomp, houts[i % e2e_slots], 0, i % e2e_slots)   # waits for the slot's previous frame
    for s_ in range(e2e_slots):
        T.tmd_host_wait(ctx, s_)
    e2e_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = n_cl_all * e2e_steps / float(te[0])
    # one frame alone (upload, decode, download back to back): the latency, not the throughput
    t0 = time.perf_counter()
    T.tmd_decode_host(ctx, hcomp, houts[0], 0, stream)
    e2e_single_s = time.perf_counter() - t0
    T.tmd_destroy(ctx)
    del h_in, keep, houts, hcomp
    torch.cuda.empty_cache()

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        peak, peak_src = (float(peaks["hbm_gbs"]), "measured") if "hbm_gbs" in peaks else (6650.0, "fallback")
        kalg = kernel_algorithmic_bytes(n_trk, n_att, n_un, geo.n_bins)
        dom = max(kms, key=kms.get)
        alg = kalg.get(dom)
        achieved = alg / (kms[dom] * 1e-3) / 1e9 if alg else None
        traffic, warp_inst, observed, src = ncu_profile_numbers(dom, args.workload)
        # second bound: instruction issue.  One warp instruction per scheduler and cycle, 4 schedulers per SM.
        props = torch.cuda.get_device_properties(device)
        sm_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0
        issue_peak = props.multi_processor_count * 4 * sm_mhz * 1e6
        second = None
        if warp_inst:
            second = {"kind": "issue", "warp_inst": warp_inst, "peak_inst_per_s": issue_peak, "sm_mhz": sm_mhz,
                      "floor_ms": 1e3 * warp_inst / issue_peak, "frac": warp_inst / (kms[dom] * 1e-3) / issue_peak,
                      "source": src}
        roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                    "frac": achieved / peak if achieved else None, "traffic": traffic, "traffic_source": src,
                    "algorithmic_bytes_per_launch": alg, "kernel_ms": kms[dom],
                    # the second bound as flat keys (nested objects do not survive every reader of this line)
                    "issue_frac": second["frac"] if second else None, "issue_floor_ms": second["floor_ms"] if second else None,
                    "bound_observed": observed, "second_bound": second,
                    "note": "kernel timed with an event pair around it in a separate pass after the timed region (same stream, "
                            "same launch configuration)"}
        st = stats(step_ms)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "ms_per_step_median": st["median"], "ms_per_step_min": st["min"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "n_tracks": n_trk, "n_attached": n_att, "n_unattached": n_un,
                       "sectors_x_rows": "36x152", "bz_tesla": BZ, "l2": "inputs larger than L2, no flush"
                       if alg_total > 400e6 else "L2-resident workload (flag)", "parallelism": f"replicas x{world}"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                    "mode": "two-slot pipeline, tmd_decode_host_async" if e2e_slots == 2 else
                    "one slot per rank (several ranks share the host's pinned memory), tmd_decode_host_async",
                    "single_frame_ms": 1e3 * e2e_single_s},
            "gpu_launches": launches,
            "clocks": clocks,
            "roofline": roofline,
            "path_gbs": alg_total / (ms_per_step * 1e-3) / 1e9, "path_frac_of_hbm_peak": alg_total / (ms_per_step * 1e-3) / 1e9 / peak,
            "kernel_ms": kms,
            "kernel_gbs": {k: kalg[k] / (kms[k] * 1e-3) / 1e9 for k in kalg if k in kms},
        }
        if world == 1 and not args.no_extras:
            other = {}
            if overlap:
                other[f"{args.workload}_two_in_flight"] = overlap
            for name in ("c2", "c4"):
                if name != args.workload:
                    other[name] = side_workload(T, name, device, min(args.steps, 10), peak)
                    torch.cuda.empty_cache()
            b = batch_workload(T, device, BATCH_FRAMES, min(args.steps, 10), peak)
            if b:
                other[f"c1x{BATCH_FRAMES}"] = b
            torch.cuda.empty_cache()
            z = entropy_workload(T, device, min(args.steps, 10), peak, args.workload)
            if z:
                other["entropy_stage"] = z
                line["e2e_container"] = z["e2e_container"]      # beside `e2e` (arrays in), which stays the headline e2e
            line["other_workloads"] = other
        if world > 1:
            line["legs_skipped"] = ["other_workloads (c2, c4, 64 x c1, two frames in flight, entropy stage): single-rank measurements",
                                    "cpu_baseline: rank 0 at N = 1 only"]
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.workload, args.cpu_tracks, device, value, not args.no_extras)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_reference(args) -> None:
    """The CPU oracle, as it stands, on bounded samples of the same workload (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import torch
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    geo, full, n_s = oracle_sample(args.workload, args.ref_tracks, dev)
    n_cl = full.n_attached + full.n_unattached
    for _ in range(args.warmup):
        time_oracle(geo, full)
    dts = [time_oracle(geo, full) for _ in range(args.steps)]
    value = n_cl * len(dts) / sum(dts)
    sample = (f"{n_s} tracks of the {args.workload} recipe ({full.n_attached} attached, {full.n_unattached} unattached) per step, "
              f"encoded by the oracle encoder; oracle/tmd_oracle.c orc_decode, single thread")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(dts) / len(dts), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "sectors_x_rows": "36x152", "bz_tesla": BZ},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "host": host_description()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c1", "c2", "c3", "c4"],
                    help="c3 = full Pb-Pb-scale time frame, the configuration the metric is quoted on")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--ref-tracks", type=int, default=25_000, help="tracks per step of the --impl reference arm")
    ap.add_argument("--cpu-tracks", type=int, default=1_000_000, help="tracks of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip other_workloads (c2, c4, 64 x c1) and the all-cores oracle run")
    ap.add_argument("--rank-logic-only", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--oracle-worker", default=None, help=argparse.SUPPRESS)
    ap.add_argument("--oracle-reps", type=int, default=1, help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.oracle_worker:
        oracle_worker(args.oracle_worker, args.oracle_reps)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(spawn_ranks(args.gpus, sys.argv[1:]))
    if args.rank_logic_only:
        run_rank_logic_only(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
