"""The seeded input generator (synth/): inputs only, no arithmetic of the method. Counter-based,
so any box, any voxel, any order gives the same values; statistics as DESIGN.md "Synthetic inputs"."""
import numpy as np

import synth


def test_boxes_voxels_and_seeds_agree():
    c = synth.Cube(123, 50, 40, 30, 7, ramp=1.0)
    full = c.fill_host()
    assert full.shape == (30, 40, 50) and full.dtype == np.float32
    box = c.fill_host(7, 5, 3, 20, 11, 9)
    assert np.array_equal(box, full[3:12, 5:16, 7:27])
    for (x, y, z) in ((0, 0, 0), (49, 39, 29), (13, 22, 8)):
        assert np.float32(c.voxel(x, y, z)) == full[z, y, x]
    assert np.array_equal(full, synth.Cube(123, 50, 40, 30, 7, ramp=1.0).fill_host(nthreads=1))
    assert not np.array_equal(full, synth.Cube(124, 50, 40, 30, 7, ramp=1.0).fill_host())


def test_noise_is_standard_normal_and_sources_are_positive():
    noise = synth.Cube(9, 96, 96, 96, 0).fill_host().astype(np.float64)
    assert abs(noise.mean()) < 5e-3 and abs(noise.std() - 1.0) < 5e-3
    assert abs((np.abs(noise) > 3).mean() - 0.0027) < 5e-4
    with_src = synth.Cube(9, 96, 96, 96, 20).fill_host().astype(np.float64)
    d = with_src - noise
    assert d.min() > -1e-5 and 3.0 < d.max() < 25.0            # peaks 3..10 sigma, may overlap


def test_nbody_kind_is_zero_background_with_halos():
    c = synth.Cube(31, 128, 96, 80, 4, kind=synth.NBODY)
    d = c.fill_host()
    assert d.min() == 0.0 and (d == 0.0).mean() > 0.2 and 0.5 <= d.max() < 4 * 30.0
    assert np.float32(c.voxel(5, 6, 7)) == d[7, 6, 5]
    assert np.array_equal(synth.Cube(31, 128, 96, 80, 4, kind=synth.SPECTRAL).fill_host(), synth.Cube(31, 128, 96, 80, 4).fill_host())
    tf = synth.tf_density()
    assert np.all(tf[:6, 3] == 0.0) and np.all(tf[6:, 3] > 0.0)
