"""Shared by the GPU parity tests: case builders and the comparison rules of DESIGN.md
"Tolerances" (north_star: 2e-3 max abs per channel in ALPHA, 1e-5 relative in MIP)."""
import numpy as np

import oracle
import synth

ALPHA_TOL = 2e-3
MIP_RTOL, MIP_ATOL = 1e-5, 1e-7


def make_pair(cube, brick, ghost=1, tf=None, tau=0.99, procedural=False, data=None):
    """(GPU volume, oracle volume) holding the same seeded cube and transfer function."""
    import torch
    import paper_1205_0282_b200 as vr
    tf = synth.tf_ramp() if tf is None else tf
    g = vr.Volume(cube.nx, cube.ny, cube.nz, brick, ghost)
    if procedural:
        o = oracle.Volume(cube.nx, cube.ny, cube.nz, brick, ghost, voxel_fn=cube.voxel_fn())
        fill_device_slabs(g, cube)
    else:
        data = cube.fill_host() if data is None else data
        o = oracle.Volume(cube.nx, cube.ny, cube.nz, brick, ghost, data=data)
        g.upload(data)
    for v in (g, o):
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(tau)
    torch.cuda.synchronize()
    return g, o


def fill_device_slabs(g, cube, slab_bytes=1 << 30):
    """Generate the cube on the device slab by slab (synth's CUDA twin) and upload each slab."""
    import torch
    plane = cube.nx * cube.ny * 4
    nzs = max(1, min(cube.nz, slab_bytes // plane))
    buf = torch.empty((nzs, cube.ny, cube.nx), dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    for z0 in range(0, cube.nz, nzs):
        nk = min(nzs, cube.nz - z0)
        part = buf[:nk]
        cube.fill_device(part.data_ptr(), 0, 0, z0, cube.nx, cube.ny, nk, st)
        g.upload(part, origin=(0, 0, z0))
    torch.cuda.synchronize()
    del buf


def gpu_frame(g, view, proj, W, H, step, mode):
    import torch
    out = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    g.render(view, proj, W, H, step, mode, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def check_alpha(gpu, ref, flags, tau, what=""):
    """gpu, ref: [...,4]; flags: oracle decision-margin flags (R12)."""
    err = np.abs(gpu - ref).max(axis=-1)
    # R14: a pixel with a sample whose NaN weight is within a factor 2 of the drop limit has two correct values
    nanm = (flags & oracle.FLAG_NAN_MARGIN) != 0
    assert nanm.mean() <= 0.01, "%s: %.2f %% of the pixels sit on the NaN-weight limit" % (what, 100 * nanm.mean())
    err = np.where(nanm, 0.0, err)
    marg = (flags & (oracle.FLAG_ERT_MARGIN | oracle.FLAG_OWNER_MARGIN)) != 0
    bad = err > np.where(marg, ALPHA_TOL + max(0.0, 1.0 - tau), ALPHA_TOL)
    assert not bad.any(), "%s ALPHA: %d pixels off, max err %.3e (unflagged max %.3e)" % (
        what, int(bad.sum()), err.max(), err[~marg].max() if (~marg).any() else 0.0)
    # R12: a ray whose opacity passes tau in steps of dA is flagged with probability ~2e-5/dA
    # (a few per cent at most); what must stay rare is a flagged pixel that really differs
    ert = (flags & oracle.FLAG_ERT_MARGIN) != 0
    assert ert.mean() < 0.03, "%s: %.4f%% early-termination-margin pixels" % (what, 100 * ert.mean())
    # owner margins (a sample within 1e-6 voxel of a brick face) are a property of the view: with the per-ray
    # step an axis-aligned ray samples ON the voxel planes; a random view has none
    assert marg.mean() < 0.10, "%s: %.4f%% decision-margin pixels" % (what, 100 * marg.mean())
    assert (err > ALPHA_TOL).mean() < 1e-3, "%s: %.4f%% pixels beyond 2e-3" % (what, 100 * (err > ALPHA_TOL).mean())
    return float(err.max())


def check_mip(gpu, ref, what="", flags=None):
    tol = MIP_RTOL * np.maximum(np.abs(gpu), np.abs(ref)) + MIP_ATOL
    err = np.abs(gpu - ref)
    if flags is not None:  # R14 / R12: pixels with two correct values (NaN-weight limit, marginal last sample)
        nanm = (flags & oracle.FLAG_NAN_MARGIN) != 0
        assert nanm.mean() <= 0.01, "%s: %.2f %% of the pixels sit on the NaN-weight limit" % (what, 100 * nanm.mean())
        loose = nanm | ((flags & oracle.FLAG_LAST_SAMPLE) != 0)
        err = np.where(loose[..., None], 0.0, err)
    bad = err > tol
    assert not bad.any(), "%s MIP: %d values off, max err %.3e" % (what, int(bad.sum()), err.max())
    return float((err / np.maximum(np.abs(ref), 1e-30)).max())


def seeded_pixels(seed, W, H, n):
    """n seeded pixels of a W x H frame (repeats are harmless)."""
    return np.array([[int(synth.u01(seed, 21, k) * W), int(synth.u01(seed, 22, k) * H)] for k in range(n)], dtype=np.int32)
