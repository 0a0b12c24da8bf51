"""Host logic: the seeded synthetic suspensions."""
import numpy as np
from scipy.spatial import cKDTree

from paper_2606_25569_b200 import inputs


def _polygon_reduced_area(P):
    x, y = P[:, 0], P[:, 1]
    xn, yn = np.roll(x, -1), np.roll(y, -1)
    A = 0.5 * abs((x * yn - xn * y).sum())
    L = np.hypot(xn - x, yn - y).sum()
    return 4 * np.pi * A / L ** 2


def test_config0_layout_and_determinism():
    a, b = inputs.config(0), inputs.config(0)
    assert a.X.shape == (16, 32, 2) and a.F.shape == (16, 32, 2) and a.mu == 1.0
    assert np.array_equal(a.X, b.X) and np.array_equal(a.F, b.F)
    c = a.X.mean(1)
    p, q = np.divmod(np.arange(16), 4)
    assert np.allclose(c, np.stack([3.0 * p, 3.0 * q], -1), atol=1e-12)
    # each vesicle is an ellipse with semi-axes (1, 0.4): extreme radii about the centre
    r = np.linalg.norm(a.X - c[:, None, :], axis=-1)
    assert np.allclose(r.max(1), 1.0, atol=1e-12) and np.allclose(r.min(1), 0.4, atol=1e-12)
    assert a.pairs == 512 * (512 - 32)


def test_config1_shapes_gap_and_area_fraction():
    s = inputs.config(1)
    assert s.X.shape == (256, 128, 2) and s.trials >= 256
    assert np.array_equal(s.X, inputs.config(1).X)
    ra = np.array([_polygon_reduced_area(P) for P in s.X])
    assert np.all(np.abs(ra - 0.65) < 2e-3)            # 128-gon of a shape tuned on a 1024-gon
    pts = s.X.reshape(-1, 2)
    pairs = cKDTree(pts).query_pairs(inputs.MIN_GAP * (1 - 1e-12), output_type="ndarray")
    ves = np.arange(len(pts)) // 128
    assert not np.any(ves[pairs[:, 0]] != ves[pairs[:, 1]])
    Lx, Ly = s.box
    assert abs(Lx - Ly) < 1e-9 and pts.min() > 0 and pts[:, 0].max() < Lx and pts[:, 1].max() < Ly
    # largest point spacing stays below the gap * sqrt(2): no crossing membranes can hide
    seg = np.linalg.norm(np.roll(s.X, -1, 1) - s.X, axis=-1)
    assert seg.max() < inputs.MIN_GAP * np.sqrt(2)
    # forces: zero-mean band-limited (k <= 16) Fourier series
    Fh = np.fft.fft(s.F, axis=1)
    assert np.abs(Fh[:, 0]).max() < 1e-9 and np.abs(Fh[:, 17:112]).max() < 1e-9


def test_channel_aspect_and_perturbation_sequence():
    s = inputs.suspension(nves=40, npts=128, phi_area=0.30, aspect=4.0, seed=7, perturb_calls=3)
    assert abs(s.box[0] / s.box[1] - 4.0) < 1e-12
    assert len(s.X_sequence) == 3 and s.X_sequence[0] is s.X
    d = s.X_sequence[1] - s.X_sequence[0]
    assert 5e-4 < d.std() < 2e-3
    assert inputs.config_shape(3) == (2000, 128) and inputs.config_shape(4) == (8000, 128)
