"""Helpers shared by the -m gpu parity tests (device buffers via PyTorch, gates of DESIGN.md)."""
import numpy as np
import torch

import oracle
from paper_1610_05801_b200 import longtrack as lt
from paper_1610_05801_b200 import workloads as wl

LAYER = 1e-4      # G17: |1 - H0/H_sep| below this = separatrix layer, gated at 1e-6
GATE = 1e-9       # BASELINE.json:north_star per-particle gate after 1000 turns
GATE_LAYER = 1e-6


def dev(a, dtype=np.float64):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def stream_ptr():
    return torch.cuda.current_stream().cuda_stream


def gpu_track(tr, z0, d0, turns, mode="fused", want_moments=False, f32=False):
    """Runs the CUDA path; returns (z, delta[, moments]) as numpy."""
    dt = np.float32 if f32 else np.float64
    z, d = dev(z0, dt), dev(d0, dt)
    n = z.numel()
    mom = None
    if mode == "fused":
        (tr.track_fused_f32 if f32 else tr.track_fused)(z, d, n, turns, stream_ptr())
    else:
        if want_moments:
            mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        (tr.track_per_turn_f32 if f32 else tr.track_per_turn)(z, d, n, turns, mom, None,
                                                              stream_ptr())
    torch.cuda.synchronize()
    out = (z.cpu().numpy(), d.cpu().numpy())
    if want_moments:
        out += (mom.cpu().numpy().view(lt.MOMENTS_DTYPE),)
    return out


def particle_errors(p, z0, d0, zg, dg, zo, do, sigma_d):
    """Normalised per-particle errors and the G17 layer mask."""
    g = oracle.derive(p)
    H0 = oracle.hamiltonian(p, z0, d0)
    layer = np.abs(1.0 - H0 / g["H_sep"]) <= LAYER
    ez = np.abs(zg - zo) / g["z_max"]
    ed = np.abs(dg - do) / sigma_d
    return ez, ed, layer


def assert_particle_gate(p, z0, d0, zg, dg, zo, do, sigma_d, gate=GATE, gate_layer=GATE_LAYER):
    ez, ed, layer = particle_errors(p, z0, d0, zg, dg, zo, do, sigma_d)
    out = ~layer
    assert out.sum() > 0
    assert ez[out].max() <= gate, "max |dz|/z_max = %.3e" % ez[out].max()
    assert ed[out].max() <= gate, "max |dd|/sigma_d = %.3e" % ed[out].max()
    if layer.any():
        assert ez[layer].max() <= gate_layer and ed[layer].max() <= gate_layer
    return dict(max_ez=float(ez[out].max()), max_ed=float(ed[out].max()), n_layer=int(layer.sum()))


def assert_moments_close(mg, mo, tol=1e-6):
    """G14: means gated against the rms, rms relative."""
    for t in range(len(mo["mean_z"])):
        assert abs(mg["mean_z"][t] - mo["mean_z"][t]) <= tol * mo["rms_z"][t], ("mean_z", t)
        assert abs(mg["mean_d"][t] - mo["mean_d"][t]) <= tol * mo["rms_d"][t], ("mean_d", t)
        assert abs(mg["rms_z"][t] / mo["rms_z"][t] - 1) <= tol, ("rms_z", t)
        assert abs(mg["rms_d"][t] / mo["rms_d"][t] - 1) <= tol, ("rms_d", t)


def count_mismatch_is_in_layer(p, zg, dg, zo, do, width=1e-6):
    """G15: where GPU and oracle disagree on membership of THEIR OWN final states, every
    such particle must sit within `width` of the separatrix (reported, not hidden)."""
    g = oracle.derive(p)
    mg, mo = oracle.bucket_mask(p, zg, dg), oracle.bucket_mask(p, zo, do)
    bad = np.where(mg != mo)[0]
    if bad.size == 0:
        return 0
    Hn = oracle.hamiltonian(p, zo[bad], do[bad]) / g["H_sep"]
    near = (np.abs(Hn - 1) < width) | (np.abs(np.abs(zo[bad]) / g["z_max"] - 1) < width)
    assert near.all(), "membership differs away from the separatrix: %s" % bad[~near][:10]
    return int(bad.size)
