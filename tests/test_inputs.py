"""The seeded generators: deterministic, the right sizes and statistics."""
import numpy as np

from paper_1601_04359_b200 import inputs


def test_configs_shapes_fractions_and_determinism():
    a = inputs.config_image(1)
    assert a.shape == (64, 64) and a.dtype == np.uint8 and set(np.unique(a)) <= {0, 1}
    assert np.array_equal(a, inputs.config_image(1))
    b = inputs.config_image(2)
    assert b.shape == (256, 256) and 0.30 <= b.mean() < 0.31
    c = inputs.config_image(3)
    assert c.shape == (512, 512) and int(c.sum()) == round(0.40 * 512 * 512)
    e = inputs.config_image(5)
    assert e.shape == (256, 256) and 0.30 <= e.mean() < 0.31 and not np.array_equal(b, e)


def test_batch_is_per_image_seeded():
    imgs = inputs.disk_batch(3, 128, 128, 6.0, 0.35, 4)
    assert imgs.shape == (3, 128, 128)
    assert np.array_equal(imgs[2], inputs.disks(128, 128, 6.0, 0.35, inputs.seed_for(4, 2)))
    assert all(0.35 <= im.mean() < 0.37 for im in imgs)
    assert not np.array_equal(imgs[0], imgs[1])


def test_gaussian_field_is_periodic_and_correlated():
    g = inputs.gaussian_field(64, 64, 4.0, 0.4, 1)
    # neighbours agree far more often than independent pixels would (2*0.4*0.6 = 0.48 disagreement)
    assert (g != np.roll(g, 1, axis=1)).mean() < 0.15
    assert (g[:, 0] != g[:, -1]).mean() < 0.2         # periodic seam is like any other column pair


def test_chess_squares_stripes():
    c = inputs.chess(20, 20, 10)
    assert c[0, 0] == 0 and c[0, 10] == 1 and c[10, 0] == 1 and c[10, 10] == 0 and c.mean() == 0.5
    s = inputs.squares(50, 50, 4, 0.2, 3)
    assert 0.2 <= s.mean() < 0.23
    h = inputs.stripes(8, 6, 4, 1, True)
    assert np.array_equal(h[:, 0], [1, 0, 0, 0, 1, 0, 0, 0])
