"""Helpers of the `-m gpu` parity tests: run the CUDA library through its C ABI on numpy inputs."""
from __future__ import annotations

import numpy as np

from tmd_inputs.layout import CLUSTER_DTYPE, COMPRESSED_FIELDS, Compressed


def gpu_decode(geo, bz, comp: Compressed, probe_step=None, flags=0, via_host=False):
    """Decode `comp` with libtmd -> (clusters[CLUSTER_DTYPE], bin_offset u32, probes u32[n_trk,6] | None)."""
    import torch
    from paper_2411_02206_b200 import tmd as T

    comp.check_shapes()
    ctx = T.tmd_create(geo, bz)
    try:
        n = comp.n_attached + comp.n_unattached
        if via_host:
            arrays = {k: np.ascontiguousarray(getattr(comp, k)) for k in COMPRESSED_FIELDS}
            clusters = np.zeros(n, CLUSTER_DTYPE)
            bin_offset = np.zeros(geo.n_bins + 1, np.uint32)
            probes = np.zeros((comp.n_tracks, 6), np.uint32) if probe_step is not None else None
            c = T.make_compressed(arrays)
            o = T.make_output(clusters, bin_offset, None, probes, T.PROBE_FINAL if probe_step is None else probe_step)
            T.tmd_decode_host(ctx, c, o, flags, 0)
            return clusters, bin_offset, probes
        dev = {}
        for k, (dt, _) in COMPRESSED_FIELDS.items():
            a = np.ascontiguousarray(getattr(comp, k))
            dev[k] = _as_torch(a).cuda()
        d_clusters = torch.full((max(n, 1) * 16,), 0xEE, dtype=torch.uint8, device="cuda")
        d_binoff = torch.zeros(geo.n_bins + 1, dtype=torch.int32, device="cuda")
        d_probe = torch.zeros(max(comp.n_tracks, 1) * 6, dtype=torch.int32, device="cuda") if probe_step is not None else None
        ws = torch.empty(T.tmd_workspace_bytes(ctx, comp.n_tracks, comp.n_attached, comp.n_unattached), dtype=torch.uint8, device="cuda")
        c = T.make_compressed(dev)
        o = T.make_output(d_clusters, d_binoff, ws, d_probe, T.PROBE_FINAL if probe_step is None else probe_step)
        stream = torch.cuda.current_stream().cuda_stream
        T.tmd_decode(ctx, c, o, flags, stream)
        torch.cuda.synchronize()
        clusters = d_clusters.cpu().numpy()[: n * 16].view(CLUSTER_DTYPE).copy()
        bin_offset = d_binoff.cpu().numpy().view(np.uint32).copy()
        probes = d_probe.cpu().numpy().view(np.uint32)[: comp.n_tracks * 6].reshape(-1, 6).copy() if d_probe is not None else None
        return clusters, bin_offset, probes
    finally:
        T.tmd_destroy(ctx)


_TORCH_VIEW = {"<u2": "int16", "i1": "int8", "u1": "uint8", "<u4": "int32"}


def _as_torch(a: np.ndarray):
    """numpy array -> torch tensor of the same width (torch lacks some unsigned dtypes; bits are what matter)."""
    import torch
    v = {"uint16": np.int16, "uint32": np.int32}.get(a.dtype.name)
    return torch.from_numpy(a.view(v) if v is not None else a)


def first_mismatch(a: np.ndarray, b: np.ndarray) -> str:
    if a.shape != b.shape:
        return f"shape {a.shape} vs {b.shape}"
    bad = np.nonzero(a != b)[0]
    if bad.size == 0:
        return "equal"
    i = int(bad[0])
    return f"{bad.size} of {a.size} differ; first at {i}: got {a[i]} want {b[i]}"
