"""The seeded input generators (SURVEY.md §8(d) recipes): shapes, determinism, rms, solenoidality."""
import numpy as np

from paper_2402_05478_b200 import inputs


def _div(v):
    nz, ny, nx = v[0].shape
    kx = np.arange(nx // 2 + 1).reshape(1, 1, -1)
    ky = np.fft.fftfreq(ny, 1.0 / ny).reshape(1, -1, 1)
    kz = np.fft.fftfreq(nz, 1.0 / nz).reshape(-1, 1, 1)
    F = [np.fft.rfftn(a) for a in v]
    return np.fft.irfftn(1j * (kx * F[0] + ky * F[1] + kz * F[2]), s=(nz, ny, nx), axes=(0, 1, 2))


def test_half_space_modes_count():
    assert len(inputs.half_space_modes(2.0)) == 16      # 32 vectors with 0<|k|<=2, one per +-k pair
    assert len(inputs.half_space_modes(1.0)) == 3


def test_config1_recipe():
    c = inputs.config1()
    assert c.shape == (32, 32, 32) and c.steps == 20 and c.cs == 1.0
    f = c.fields
    b2 = np.mean(f["bx"] ** 2 + f["by"] ** 2 + f["bz"] ** 2)
    assert abs(np.sqrt(b2) - 0.1) < 1e-14
    assert np.max(np.abs(_div([f["bx"], f["by"], f["bz"]]))) < 1e-13
    assert abs(np.mean(f["rho"]) - 1.0) < 1e-15 and 0.9 < f["rho"].min()
    assert abs(np.mean(f["ux"] ** 2 + f["uy"] ** 2 + f["uz"] ** 2) - 3.0) < 1e-13   # ABC, A=B=C=1
    d = inputs.config1()
    assert all(np.array_equal(a, b) for a, b in zip(c.arrays(), d.arrays()))          # seeded


def test_config2_and_3_recipes():
    c = inputs.config2(64, 10)
    assert c.shape == (1, 64, 64) and c.hydro and c.cs == 2.0
    assert np.max(np.abs(c.fields["uy"])) < 5e-3 and not np.any(c.fields["bx"])
    c = inputs.config3(16, 5)
    assert abs(np.mean(c.fields["bx"] ** 2) - 0.5) < 1e-14 and not np.any(c.fields["uz"])


def test_config4_recipe_small():
    c = inputs.config4(48, 3)
    f = c.fields
    assert abs(np.sqrt(np.mean(f["ux"] ** 2 + f["uy"] ** 2 + f["uz"] ** 2)) - 1.0) < 1e-13
    assert abs(np.sqrt(np.mean(f["bx"] ** 2 + f["by"] ** 2 + f["bz"] ** 2)) - 0.5) < 1e-13
    assert np.max(np.abs(_div([f["ux"], f["uy"], f["uz"]]))) < 1e-11
    spec = np.abs(np.fft.rfftn(f["ux"]))
    assert spec[20:30, 20:30, 17:].max() < 1e-9 * spec.max()          # nothing beyond the mask (kcut = 15)
    assert inputs.config5_batch(8).shape == (7, 8, 8, 8)
