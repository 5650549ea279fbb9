"""Seeded input generators: determinism and the structure DESIGN.md's input recipe states.  CPU only."""
import numpy as np

import lbm_inputs as I


def test_generators_are_deterministic():
    a = I.make_config(3, shape=(32, 48, 96))
    b = I.make_config(3, shape=(32, 48, 96))
    assert np.array_equal(a["flags"], b["flags"]) and np.array_equal(a["d"], b["d"])
    u1 = I.spectral_field((16, 16, 16), 4, 32, 0.03, seed=5)
    u2 = I.spectral_field((16, 16, 16), 4, 32, 0.03, seed=5)
    assert np.array_equal(u1, u2)


def test_spectral_field_is_the_stated_fourier_sum():
    shape = (12, 10, 8)
    nz, ny, nx = shape
    u = I.spectral_field(shape, 3, 16, 0.03, seed=9)
    assert abs(np.sqrt((u ** 2).sum(axis=0).mean()) - 0.03) < 1e-15
    k, e, ph, amp = I.spectral_modes(3, 16, seed=9)
    assert np.abs((k * e).sum(axis=1)).max() < 1e-12          # divergence-free polarisation
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ref = np.zeros((3,) + shape)
    for m in range(16):
        arg = 2 * np.pi * (k[m, 0] * x / nx + k[m, 1] * y / ny + k[m, 2] * z / nz) + ph[m]
        ref += amp[m] * e[m][:, None, None, None] * np.cos(arg)
    ref *= 0.03 / np.sqrt((ref ** 2).sum(axis=0).mean())
    assert np.abs(u - ref).max() < 1e-14


def test_urban_channel_structure():
    nz, ny, nx = 64, 96, 192
    flags, d = I.urban_channel(nx, ny, nz, seed=1003)
    t = flags & 0x0F
    assert (t[0] == I.SOLID).all() and (t[nz - 1] == I.SOLID).all()
    assert (t[1:nz - 1, :, 0] == I.INLET).all() and (t[1:nz - 1, :, nx - 1] == I.OUTLET).all()
    assert set(np.unique(flags)) <= {0, 1, 2, 3, I.WM_FLOOR}
    build = (d == 1.0) & (t == I.FLUID)
    assert build[1].mean() >= 0.15 * 0.95                       # footprint cover
    trees = (d > 0) & (d < 1)
    assert trees.mean() >= 0.05
    assert d[trees].min() >= 0.2 and d[trees].max() <= 0.6
    wm = flags == I.WM_FLOOR
    assert wm[1].any() and not wm[2:].any() and (d[wm] == 1.0).all()
    # keep-out zones are free of obstacles
    assert not (d[2:, :, : nx // 12] > 0).any() and not (d[2:, :, nx - nx // 6:] > 0).any()


def test_random_spheres_fraction():
    flags = I.random_spheres((48, 48, 48), seed=1004)
    frac = (flags == I.SOLID).mean()
    assert 0.10 <= frac < 0.16


def test_config_table():
    c1 = I.make_config(1)
    assert c1["Q"] == 19 and c1["dtype"] == "f64" and c1["shape"] == (32, 32, 32) and c1["steps"] == 100
    c2 = I.make_config(2, shape=(32, 32, 32), k_max=4, n_modes=32)
    assert abs(c2["params"]["tau0"] - 0.50003) < 1e-12 and c2["params"]["cs_smago"] == 0.1
    c4 = I.make_config(4, shape=(48, 48, 48), k_max=4, n_modes=32)
    assert c4["Q"] == 27 and np.abs(c4["u"][:, c4["flags"] == I.SOLID]).max() == 0.0


def test_config8_wall_model_cells_on_building_faces_point_away_from_the_face():
    cfg = I.make_config(8, shape=(40, 48, 160))
    base = I.make_config(7, shape=(40, 48, 160))
    fl, d = cfg["flags"], cfg["d"]
    building = (base["d"] == 1.0) & ((base["flags"] & 15) == I.FLUID)
    new = ((fl & 15) == I.WALLMODEL) & ((base["flags"] & 15) != I.WALLMODEL)
    assert new.sum() == sum(cfg["wm_face_cells"].values()) > 1000
    assert (base["d"][new] == 0.0).all() and (d[new] == 1.0).all()
    # the cell behind every new wall-model cell (x - n) is a building cell
    for z, y, x in np.argwhere(new)[::7]:
        code = fl[z, y, x] >> 4
        n = [0, 0, 0]
        n[code >> 1] = -1 if (code & 1) else 1
        assert building[z - n[2], y - n[1], x - n[0]]
    # ... and the cell in front of it (x + n, where the wall model samples the velocity) is plain fluid
    for z, y, x in np.argwhere(new)[::5]:
        code = fl[z, y, x] >> 4
        n = [0, 0, 0]
        n[code >> 1] = -1 if (code & 1) else 1
        assert fl[z + n[2], y + n[1], x + n[0]] == I.FLUID and d[z + n[2], y + n[1], x + n[0]] == 0.0
    # nothing else changed
    assert np.array_equal(fl[~new], base["flags"][~new]) and np.array_equal(d[~new], base["d"][~new])
