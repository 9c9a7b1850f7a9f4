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


def _expand(mask, like):
    return mask.reshape(mask.shape + (1,) * (like.ndim - mask.ndim))


def _best_over_candidates(gpu, ref, key, errfn, want_ert, want_nan, envelope=False):
    """R12: a decision-margin pixel has several correct values - the oracle's with each marginal decision taken
    either way (early-termination tests within 1e-5 of tau: tau -/+ 1e-5; samples whose NaN weight is within a
    factor 2 of R14's limit: limit x 0.5 / x 2). Returns, per pixel, the smallest error over those candidates;
    the caller applies it to flagged pixels only and holds it to the NORMAL tolerance."""
    best = errfn(gpu, ref[key])
    m = ref.get("ert_margin", 1e-5)
    cands = [ref[key]]
    for dtau in ((0.0, -m, m) if want_ert else (0.0,)):
        for ns in ((1.0, 0.5, 2.0) if want_nan else (1.0,)):
            if dtau == 0.0 and ns == 1.0:
                continue
            cands.append(ref["alt"](dtau, ns)[key])
            best = np.minimum(best, errfn(gpu, cands[-1]))
    if envelope and len(cands) > 1:
        # a ray that stops anywhere between the two extreme decisions lies, channel by channel, between their
        # results (premultiplied colour and opacity only grow along a ray): distance to that interval
        lo, hi = np.minimum.reduce(cands), np.maximum.reduce(cands)
        best = np.minimum(best, np.maximum(np.maximum(lo - gpu, gpu - hi), 0.0).max(axis=-1))
    return best


def check_alpha(gpu, ref, tau, what="", key="image", envelope=False, max_flagged=0.10):
    """gpu: [...,4]; ref: the oracle's result dict for the same pixels (image / sub, flags, alt)."""
    flags = ref["flags"]
    want = ref[key]
    if want.ndim > flags.ndim + 1:          # sub-images [npix][nbricks][4]: the pixel's flags apply to each brick
        flags = _expand(flags, want[..., 0])
        flags = np.broadcast_to(flags, want.shape[:-1])

    def errfn(a, b):
        return np.abs(a - b).max(axis=-1)

    err = errfn(gpu, want)
    ert = (flags & oracle.FLAG_ERT_MARGIN) != 0
    nanm = (flags & oracle.FLAG_NAN_MARGIN) != 0
    loose = ert | nanm
    if loose.any():  # flagged pixels are CHECKED, against every candidate, at the normal tolerance (not excused)
        err = np.where(loose, _best_over_candidates(gpu, ref, key, errfn, ert.any(), nanm.any(), envelope), err)
    # owner-margin pixels (FLAG_OWNER_MARGIN) get no allowance: both sides take the owner decision in FP64 with the
    # same operations, so the sample sets are identical
    bad = err > ALPHA_TOL
    assert not bad.any(), "%s ALPHA: %d pixels off, max err %.3e (unflagged max %.3e)" % (
        what, int(bad.sum()), err.max(), err[~loose].max() if (~loose).any() else 0.0)
    # R12: a (ray, brick) whose opacity passes tau in steps of dA is flagged with probability ~2e-5/dA (1-2 % on the
    # ramp), a pixel if any of the bricks its ray saturates is (measured: up to 6.5 % of a block of c3 pixels that all hit
    # the cube). Flagged pixels are checked above like the others, so this is a sanity bound on the flag, not an allowance.
    assert ert.mean() < max_flagged, "%s: %.4f%% early-termination-margin pixels" % (what, 100 * ert.mean())
    assert nanm.mean() <= 0.01, "%s: %.2f %% of the pixels sit on the NaN-weight limit" % (what, 100 * nanm.mean())
    return float(err.max())


def check_mip(gpu, ref, what="", key="image"):
    """ref: the oracle's result dict, or a plain array (comparisons between two GPU frames)."""
    want = ref[key] if isinstance(ref, dict) else ref

    def errfn(a, b):
        return (np.abs(a - b) - (MIP_RTOL * np.maximum(np.abs(a), np.abs(b)) + MIP_ATOL)).max(axis=-1)

    excess = errfn(gpu, want)  # <= 0 where within R13's tolerance
    if isinstance(ref, dict):
        # FLAG_LAST_SAMPLE pixels get no allowance: the existence of the clipped last sample is decided in FP64 on both
        # sides. R14: a sample on the NaN-weight limit may be kept or dropped - both candidates are tried.
        nanm = (ref["flags"] & oracle.FLAG_NAN_MARGIN) != 0
        assert nanm.mean() <= 0.01, "%s: %.2f %% of the pixels sit on the NaN-weight limit" % (what, 100 * nanm.mean())
        if nanm.any():
            excess = np.where(nanm, _best_over_candidates(gpu, ref, key, errfn, False, True), excess)
    bad = excess > 0.0
    assert not bad.any(), "%s MIP: %d pixels off, max excess over tolerance %.3e" % (what, int(bad.sum()), excess.max())
    return float((np.abs(gpu - want) / np.maximum(np.abs(want), 1e-30)).max())


def seeded_pixels(seed, W, H, n):
    """n seeded pixels of a W x H frame (repeats are harmless)."""
    return np.array([[int(synth.u01(seed, 21, k) * W), int(synth.u01(seed, 22, k) * H)] for k in range(n)], dtype=np.int32)
