"""vr_composite_static: stand-alone compositing (row a9) without any allocation - the two device tables live in a fixed
__device__ array inside libvr (include/vr.h). Checked against the existing path (vr_composite, same kernel: bit-identical)
and against the oracle at R15's 1e-5, on two calls in a row that share the array (the second with other layers, another
order and FEWER layers, so stale entries of the first call are there to be misread), and for the size limit.
Collected last on purpose (file name): a failure here must not hide another test under `pytest -x`."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vr(cuda_device):
    from paper_1205_0282_b200 import build
    build.build()
    import paper_1205_0282_b200 as vr
    return vr


def _layers(seed, n, W, H):
    rects, layers_h = [], []
    for l in range(n):
        x0, y0 = int(synth.u01(seed, 1, l) * W * 0.6), int(synth.u01(seed, 2, l) * H * 0.6)
        x1 = min(W, x0 + 5 + int(synth.u01(seed, 3, l) * W * 0.7))
        y1 = min(H, y0 + 3 + int(synth.u01(seed, 4, l) * H * 0.8))
        if l == 0:
            x0, y0, x1, y1 = 0, 0, W, H
        if l == 1:
            x1 = x0  # an empty layer
        rects.append((x0, y0, x1, y1))
        layers_h.append(synth.layer_host(seed + 90, l, 0, (x1 - x0) * (y1 - y0)).reshape(y1 - y0, x1 - x0, 4))
    return rects, layers_h, synth.permutation(seed + 4, n)


def test_composite_static_matches_the_allocating_path_twice_in_a_row(vr):
    import torch
    W, H = 203, 117
    frames = []
    for call, (seed, n) in enumerate(((3, 40), (8, 11))):
        rects, layers_h, order = _layers(seed, n, W, H)
        layers_d = [torch.from_numpy(l).cuda() if l.size else torch.empty((0, 0, 4), device="cuda") for l in layers_h]
        want = torch.full((H, W, 4), 7.0, dtype=torch.float32, device="cuda")
        got = torch.full((H, W, 4), -3.0, dtype=torch.float32, device="cuda")
        vr.composite(layers_d, rects, order, W, H, want)
        vr.composite_static(layers_d, rects, order, W, H, got)
        torch.cuda.synchronize()
        got_h = got.cpu().numpy()
        assert np.array_equal(got_h, want.cpu().numpy()), "call %d: differs from vr_composite" % call
        assert np.abs(got_h - oracle.composite(layers_h, rects, order, W, H)).max() < 1e-5  # R15
        frames.append(got_h)
    assert np.abs(frames[0] - frames[1]).max() > 1e-2  # two different frames went through the one array


def test_composite_static_limit_and_errors(vr):
    import torch
    W, H = 64, 48
    nmax = vr.COMPOSITE_STATIC_MAX_LAYERS
    layer = torch.full((H, W, 4), 0.001, dtype=torch.float32, device="cuda")
    out = torch.zeros((H, W, 4), dtype=torch.float32, device="cuda")
    ref = torch.zeros((H, W, 4), dtype=torch.float32, device="cuda")
    rect = (0, 0, W, H)
    # exactly the maximum: allowed, and equal to the allocating path
    vr.composite_static([layer] * nmax, [rect] * nmax, np.arange(nmax), W, H, out)
    vr.composite([layer] * nmax, [rect] * nmax, np.arange(nmax), W, H, ref)
    torch.cuda.synchronize()
    assert torch.equal(out, ref) and float(out[..., 3].min()) > 0.2
    # one more: refused with a message that names the limit, output untouched
    out.fill_(5.0)
    with pytest.raises(vr.VrError) as err:
        vr.composite_static([layer] * (nmax + 1), [rect] * (nmax + 1), np.arange(nmax + 1), W, H, out)
    assert str(nmax) in str(err.value)
    with pytest.raises(vr.VrError):
        vr.composite_static([layer] * 3, [rect] * 3, np.zeros(3, dtype=np.int32), W, H, out)  # not a permutation
    torch.cuda.synchronize()
    assert float(out.min()) == 5.0 and float(out.max()) == 5.0
    # no layers at all: a cleared frame
    vr.composite_static([], np.zeros((0, 4), dtype=np.int32), np.zeros(0, dtype=np.int32), W, H, out)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
