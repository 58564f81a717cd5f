"""The seeded input generators: determinism, shapes, packing.  CPU only."""
import hashlib

import numpy as np

from workloads import CONFIGS, default_rho, scaled_rho, make_workload, pack_mask, splitmix64, uniform01, weight_grid


def test_splitmix64_reference_values():
    # published SplitMix64 test vector: seed 0 -> first outputs
    out = splitmix64(0, np.arange(3))
    assert [int(x) for x in out] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    u = uniform01(12345, np.arange(1000))
    assert u.min() >= 0.0 and u.max() < 1.0 and abs(u.mean() - 0.5) < 0.05


def test_config0_shapes_and_determinism():
    a = make_workload(0); b = make_workload(0)
    assert (a.N, a.n, a.B) == (3000, 240, 9)
    assert a.phi.dtype == np.float32 and a.phi.flags.c_contiguous
    assert np.array_equal(a.phi, b.phi) and np.array_equal(a.points, b.points)
    assert (a.point_class == 0).sum() == 1000 and (a.point_class == 1).sum() == 2000
    r = np.linalg.norm(a.points, axis=1)
    assert r[:1000].max() <= 5.0 and r[1000:].min() >= 7.0 and r[1000:].max() <= 15.0
    assert np.linalg.norm(a.isocenters, axis=1).max() <= 5.0
    # column order j = (iso*8 + sector)*3 + collimator ; entries a_s * exp(-d^2 / (2 sigma^2))
    i, iso, s, c = 17, 4, 5, 1
    d2 = np.sum((a.points[i] - a.isocenters[iso]) ** 2)
    g = a.phi[i, (iso * 8 + s) * 3 + c] / np.exp(-d2 / (2 * 4.0 ** 2))
    assert 0.8 <= g <= 1.2
    assert np.allclose(a.phi[:, (iso * 8 + s) * 3 + 0] / np.float32(g), np.exp(-np.sum((a.points - a.isocenters[iso]) ** 2, axis=1) / 8.0), rtol=1e-5, atol=1e-30)
    assert list(a.weights[5]) == [1.0, 0.5, 1.0]       # p = i_alpha*3 + i_beta


def test_grids_and_rho_rule():
    al, be, w = weight_grid(21)
    assert w.shape == (441, 3) and np.isclose(be[1], 0.05) and np.isclose(al[21], 0.05)
    rho = default_rho(be, rho0=1e-3)
    assert np.isclose(rho[0], 1e-3) and np.isclose(rho[1], 1e-3) and np.isclose(rho[20], 1e-3 * np.sqrt(0.05))
    for k, spec in CONFIGS.items():
        assert spec["n_iso"] * 24 in (240, 1440, 9600, 12000)
    # size-aware rule: identical to default_rho at config 0's N_T = 1000 for beta >= beta0, 256x at beta = 0
    pc = np.array([0] * 1000 + [1] * 2000, dtype=np.uint8)
    rs = scaled_rho(be, pc)
    assert np.allclose(rs[1:21], rho[1:21]) and np.isclose(rs[0], 0.256)
    assert np.allclose(scaled_rho(be, np.repeat(pc, 20)), rs / 20)


def test_masks_and_multitarget_small():
    w = make_workload(2, n_target=900, n_lowdose=1800, n_iso=18, grid=3)
    assert w.n == 18 * 24 and w.N == 2700 and w.B == 9
    assert w.row_mask.shape == (9, (2700 + 31) // 32) and w.row_mask.dtype == np.uint32
    mb = w.mask_bool()
    assert mb[:, :900].all()                               # target rows always active
    frac = mb[:, 900:].mean(axis=1)
    assert np.all(frac > 0.75) and np.all(frac <= 1.0) and frac.std() > 0.01
    assert np.array_equal(pack_mask(mb), w.row_mask)
    assert len(w.radii) == 9 and abs(np.sum(4 / 3 * np.pi * w.radii ** 3) - 52000.0) < 1e-6
    d = np.linalg.norm(w.centres[:, None] - w.centres[None], axis=2) + 1e9 * np.eye(9)
    assert d.min() >= 25.0
    h = hashlib.sha256(w.phi.tobytes()).hexdigest()
    assert h == hashlib.sha256(make_workload(2, n_target=900, n_lowdose=1800, n_iso=18, grid=3).phi.tobytes()).hexdigest()
