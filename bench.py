#!/usr/bin/env python
"""bench.py -- decoded TPC clusters/s of the track-model decoder on synthetic time frames (BASELINE.json metric).

One "step" = one pass of the whole hot path over one synthetic time frame:
`tmd_decode` through the C ABI, compressed SoA resident in HBM.  Prints ONE JSON line (see the task contract):
value = clusters decoded per second over all ranks (device-timed with CUDA events, max over ranks), `e2e` = the same
through `tmd_decode_host` with pinned HOST buffers (copies inside the timed region), `roofline` for the dominant kernel
(timed live with CUDA events the library records on the launching stream), `cpu_baseline` = the CPU oracle on a bounded
sample of the same workload.

Multi-GPU: the path does not shard ("replicas only") -- every rank decodes its own time frame
(different seed), no collective on the data path; torch.distributed (NCCL) is used for the barrier and the max.

`--impl reference` times the CPU oracle (oracle/, as it stands, single thread) on bounded samples of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

BZ = 0.5
METRIC = "decoded_tpc_clusters_per_second"
UNIT = "clusters/s"


def algorithmic_bytes_attached(n_trk: int, n_att: int) -> int:
    """per-track 11 B + copy-through 7 B/cluster + residual streams 8 B/residual in, 16 B/cluster out."""
    return 11 * n_trk + 7 * n_att + 8 * (n_att - n_trk) + 16 * n_att


def algorithmic_bytes_unattached(n_un: int, n_bins: int) -> int:
    return 13 * n_un + 4 * n_bins + 16 * n_un + 4 * (n_bins + 1)


def kernel_algorithmic_bytes(n_trk: int, n_att: int, n_un: int, n_bins: int) -> dict:
    """The share of the algorithmic bytes each kernel is there to move: the decode kernel consumes the
    per-track fields and the four residual streams, the scatter kernel the copy-through fields and writes the records,
    the unattached kernel its 13 B in / 16 B out.  The walk/rank and scan kernels move no algorithmic byte (overhead)."""
    return {"track_decode": 11 * n_trk + 8 * (n_att - n_trk), "scatter": 7 * n_att + 16 * n_att,
            "unattached": algorithmic_bytes_unattached(n_un, n_bins)}


# ------------------------------------------------------------------------------------------------ workload on the device
def build_workload(name: str, device, seed_offset: int = 0, keep_truth: bool = False):
    """Synthetic time frame `name` (tmd_inputs.timeframe.WORKLOADS) as device tensors of the compressed SoA.
    Attached clusters: helix truth -> the library's own encoder (tmd_encode_attached); unattached: compressed domain."""
    import torch
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs import build_geometry, timeframe as tf

    geo = build_geometry(36)
    mk, n_un, single = tf.WORKLOADS[name]
    cfg = mk()
    cfg.seed += 1000 * seed_offset
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
    T.tmd_destroy(ctx)
    del ws
    if not keep_truth:
        truth = None
    arrays.update(tf.generate_unattached(geo, n_un, cfg.seed, device, "inv_x", single))
    torch.cuda.empty_cache()
    return (geo, arrays, truth) if keep_truth else (geo, arrays)


def oracle_sample(workload: str, n_s: int, device):
    """A bounded sample of `workload` for the CPU oracle: the first n_s tracks of the same generator recipe (same pT / length /
    looper mix) and the same fraction of the unattached clusters.  The attached clusters are ENCODED BY THE ORACLE'S OWN
    ENCODER -- nothing the oracle reads comes from the CUDA path."""
    import torch
    from tmd_inputs import build_geometry, physical as ph, timeframe as tf
    from tmd_inputs.layout import COMPRESSED_FIELDS, Compressed
    from oracle import tmd_oracle as O

    geo = build_geometry(36)
    mk, n_un, single = tf.WORKLOADS[workload]
    cfg = mk()
    n_s = min(cfg.n_tracks, n_s)
    frac = n_s / cfg.n_tracks
    cfg.n_tracks = n_s
    tr = tf.generate_truth(cfg, geo, device, batch=400_000)
    ev_att = tr.att.cpu().numpy().view(ph.CLUSTER_DTYPE).reshape(-1)
    comp = O.encode(geo, BZ, tr.trk_ncl.cpu().numpy().view(np.uint16), tr.trk_qptf.cpu().numpy(), ev_att, tr.leg.cpu().numpy(),
                    np.zeros(0, ph.CLUSTER_DTYPE))
    del tr, ev_att
    u = tf.generate_unattached(geo, int(n_un * frac), cfg.seed, device, "inv_x", single)
    full = Compressed.empty(comp.n_tracks, comp.n_attached, int(u["u_qtot"].shape[0]), geo.n_bins)
    for k, (dt, _) in COMPRESSED_FIELDS.items():
        src = u[k].cpu().numpy().view(np.dtype(dt)) if k in u else getattr(comp, k)
        getattr(full, k)[:] = src
    return geo, full, n_s


def time_oracle(geo, comp) -> float:
    from oracle import tmd_oracle as O
    t0 = time.perf_counter()
    O.decode(geo, BZ, comp)
    return time.perf_counter() - t0


def cpu_baseline(workload: str, n_s: int, device) -> dict:
    """The oracle as it stands (single thread) timed on a bounded sample of the workload (about 10 s of decoding at c3)."""
    geo, comp, n_s = oracle_sample(workload, n_s, device)
    dt = time_oracle(geo, comp)
    n_cl = comp.n_attached + comp.n_unattached
    return {"value": n_cl / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{n_s} tracks of the {workload} recipe ({comp.n_attached} attached) + the same fraction of the unattached "
                      f"clusters ({comp.n_unattached}), encoded by the oracle encoder; oracle/tmd_oracle.c orc_decode, single "
                      f"thread, {dt:.2f} s"}


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


# ------------------------------------------------------------------------------------------------ arms
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


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist
    from paper_2411_02206_b200 import tmd as T

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)

    geo, arrays = build_workload(args.workload, device, seed_offset=rank_seed_offset(rank))
    n_trk, n_att, n_un = (int(arrays[k].shape[0]) for k in ("trk_ncl", "a_qtot", "u_qtot"))
    n_cl = n_att + n_un
    ctx = T.tmd_create(geo, BZ)
    clusters = torch.empty(n_cl * 16, dtype=torch.uint8, device=device)
    bin_offset = torch.empty(geo.n_bins + 1, dtype=torch.int32, device=device)
    ws = torch.empty(T.tmd_workspace_bytes(ctx, n_trk, n_att, n_un), dtype=torch.uint8, device=device)
    comp = T.make_compressed(arrays)
    out = T.make_output(clusters, bin_offset, ws)
    stream = torch.cuda.current_stream().cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        T.tmd_decode(ctx, comp, out, 0, stream)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ktimes: dict[str, float] = {}
    launches = 0
    for s0, s1 in ev:
        s0.record()
        T.tmd_decode(ctx, comp, out, T.TMD_TIMING, stream)
        s1.record()
        launches += T.tmd_last_launch_count(ctx)
        for name, ms in T.tmd_kernel_times(ctx):          # waits for this step's last kernel
            ktimes[name] = ktimes.get(name, 0.0) + ms
    barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    total_ms, n_cl_all = aggregate_over_ranks(total_ms, float(n_cl), device)
    ms_per_step = total_ms / args.steps
    value = n_cl_all / (ms_per_step * 1e-3)
    # ---- outside the timed region: the same step with every kernel alone on one stream (TMD_SERIAL), for the
    #      per-kernel times without overlap that the roofline of the dominant kernel is computed from
    kserial: dict[str, float] = {}
    n_serial = 3
    for _ in range(n_serial):
        T.tmd_decode(ctx, comp, out, T.TMD_TIMING | T.TMD_SERIAL, stream)
        for name, ms in T.tmd_kernel_times(ctx):
            kserial[name] = kserial.get(name, 0.0) + ms / n_serial
    torch.cuda.synchronize()

    # ---- end to end: pinned host buffers in, pinned host buffers out, every copy inside the timed region.  Frames go
    #      through the library's two-slot pipeline (tmd_decode_host_async): the upload of frame i+1 runs beside the
    #      download of frame i, as in the paper's deployment; each slot has its own output buffers.
    h_in = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in arrays.items()}
    h2d = sum(v.numel() * v.element_size() for v in h_in.values())
    del clusters, ws
    torch.cuda.empty_cache()
    hcomp = T.make_compressed(h_in)
    houts, keep = [], []
    for _ in range(T.TMD_HOST_SLOTS):
        hc = torch.empty(n_cl * 16, dtype=torch.uint8, pin_memory=True)
        hb = torch.empty(geo.n_bins + 1, dtype=torch.int32, pin_memory=True)
        keep.append((hc, hb))
        houts.append(T.make_output(hc, hb))
    d2h = keep[0][0].numel() + keep[0][1].numel() * 4
    e2e_steps = max(2, min(args.steps, args.e2e_steps))
    for s_ in range(T.TMD_HOST_SLOTS):                        # warm-up: allocates the slots' device arenas
        T.tmd_decode_host_async(ctx, hcomp, houts[s_], 0, s_)
    for s_ in range(T.TMD_HOST_SLOTS):
        T.tmd_host_wait(ctx, s_)
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        T.tmd_decode_host_async(ctx, hcomp, houts[i % T.TMD_HOST_SLOTS], 0, i % T.TMD_HOST_SLOTS)   # waits for the slot's previous frame
    for s_ in range(T.TMD_HOST_SLOTS):
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

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        peak, peak_src = (float(peaks["hbm_gbs"]), "measured") if "hbm_gbs" in peaks else (6650.0, "fallback")
        kavg = {k: v / args.steps for k, v in ktimes.items()}
        kalg = kernel_algorithmic_bytes(n_trk, n_att, n_un, geo.n_bins)
        dom = max(kserial, key=kserial.get)
        alg = kalg.get(dom)
        achieved = alg / (kserial[dom] * 1e-3) / 1e9 if alg else None
        roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                    "frac": achieved / peak if achieved else None, "traffic": ncu_traffic(dom, args.workload),
                    "algorithmic_bytes_per_launch": alg, "kernel_ms": kserial[dom],
                    "kernel_ms_in_timed_region": kavg.get(dom),
                    "note": "kernel timed alone on one stream (TMD_SERIAL pass after the timed region); in the timed region "
                            "it shares the GPU with the unattached kernel of the second stream"}
        total_alg = algorithmic_bytes_attached(n_trk, n_att) + algorithmic_bytes_unattached(n_un, geo.n_bins)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": args.workload, "n_tracks": n_trk, "n_attached": n_att, "n_unattached": n_un,
                       "sectors_x_rows": "36x152", "bz_tesla": BZ, "l2": "inputs larger than L2, no flush"
                       if total_alg > 400e6 else "L2-resident workload (flag)", "parallelism": f"replicas x{world}"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                    "mode": "two-slot pipeline, tmd_decode_host_async", "single_frame_ms": 1e3 * e2e_single_s},
            "gpu_launches": launches,
            "clocks": clocks,
            "roofline": roofline,
            "path_gbs": total_alg / (ms_per_step * 1e-3) / 1e9, "path_frac_of_hbm_peak": total_alg / (ms_per_step * 1e-3) / 1e9 / peak,
            "kernel_ms": kavg, "kernel_ms_serial": kserial,
            "kernel_gbs_serial": {k: kalg[k] / (kserial[k] * 1e-3) / 1e9 for k in kalg if k in kserial},
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.workload, args.cpu_tracks, device)
        print(json.dumps(line), flush=True)
    T.tmd_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()


def ncu_traffic(kernel: str, workload: str):
    """dram bytes per launch of `kernel` from the committed ncu summary (profiles/traffic.txt), else None."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "traffic.txt")):
            v = line.split()
            if len(v) >= 3 and v[0] == workload and v[1] == kernel:
                return float(v[2])
    except OSError:
        pass
    return None


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
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
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
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
