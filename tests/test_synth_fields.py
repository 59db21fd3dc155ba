"""The seeded input generators (synth/): properties that the recipe of DESIGN.md section 4 states.  No method arithmetic here."""
import numpy as np
import pytest

import synth


def _plaquette(U):
    s, n = 0.0, 0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a = U[..., mu, :, :]
            b = np.roll(U[..., nu, :, :], -1, axis=mu)
            c = np.roll(U[..., mu, :, :], -1, axis=nu)
            d = U[..., nu, :, :]
            p = a @ b @ np.conj(np.swapaxes(c, -1, -2)) @ np.conj(np.swapaxes(d, -1, -2))
            s += np.trace(p, axis1=-2, axis2=-1).real.mean() / 3
            n += 1
    return s / n


@pytest.mark.parametrize("gen", ["white", "smooth"])
def test_links_are_su3_and_reproducible(gen):
    dims = (8, 4, 8, 4)
    make = (lambda: synth.su3_links(dims, 0.3, 1)) if gen == "white" else (lambda: synth.su3_links_smooth(dims, 0.7, 1, 4))
    U = make()
    assert U.shape == dims + (4, 3, 3) and U.dtype == np.complex128
    V = U.reshape(-1, 3, 3)
    assert np.abs(V @ np.conj(np.swapaxes(V, 1, 2)) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(V) - 1.0).max() < 1e-13
    assert np.array_equal(U, make())                      # a pure function of (seed, site, direction)


def test_smooth_links_have_long_range_order():
    """su3_links_smooth: generators drawn every `corr` sites and interpolated.  At the SAME eps the plaquette is much closer to 1
    than for the white-noise field, neighbouring links are close, corr = 1 reproduces independent links, and extents that are
    not multiples of corr are rejected."""
    dims = (8, 8, 8, 8)
    white = synth.su3_links(dims, 0.7, 1)
    smooth = synth.su3_links_smooth(dims, 0.7, 1, 4)
    pw, ps = _plaquette(white), _plaquette(smooth)
    assert ps > 0.7 and pw < 0.2 and ps > pw + 0.5, (pw, ps)
    d_s = np.abs(smooth - np.roll(smooth, 1, axis=0)).mean()
    d_w = np.abs(white - np.roll(white, 1, axis=0)).mean()
    assert d_s < 0.35 * d_w
    assert _plaquette(synth.su3_links_smooth(dims, 0.7, 1, 1)) < 0.2     # no interpolation: white noise again
    assert not np.array_equal(smooth, synth.su3_links_smooth(dims, 0.7, 2, 4))
    with pytest.raises(ValueError):
        synth.su3_links_smooth((8, 8, 6, 8), 0.7, 1, 4)
