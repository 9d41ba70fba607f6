"""Comparison metrics for the GPU-vs-oracle parity tests (SURVEY.md 8(c) reading A19)."""
import numpy as np

TOL_SITE = {"f64": 1e-12, "f32": 2e-5}        # BASELINE.json:north_star
TOL_SUM = {"f64": 1e-10, "f32": 1e-5}         # fp64: north_star; fp32: DESIGN.md "Tolerances"


def site_rel_err(got: np.ndarray, want: np.ndarray, per: int = 1) -> np.ndarray:
    """e(x) = ||got(x) - want(x)||_F / max(||want(x)||_F, 1e-300) over the site's record.
    `per` trailing axes... records: got/want [V, ...] -> one number per leading entry;
    for a gauge field pass arrays reshaped to [V*4, 3, 3] to get one number per link."""
    g = got.reshape(got.shape[0], -1).astype(np.complex128)
    w = want.reshape(want.shape[0], -1).astype(np.complex128)
    num = np.sqrt((np.abs(g - w) ** 2).sum(axis=1))
    den = np.maximum(np.sqrt((np.abs(w) ** 2).sum(axis=1)), 1e-300)
    return num / den


def links(u: np.ndarray) -> np.ndarray:
    return u.reshape(-1, 3, 3)


def z3_fix(got_links: np.ndarray, want_links: np.ndarray, theta: np.ndarray | None = None):
    """A9: where the determinant phase sits on the branch cut the two sides may differ by
    a centre element exp(+-2 pi i/3); returns got with the best centre element applied
    and the number of links where a non-trivial one was needed."""
    z = np.exp(2j * np.pi * np.arange(3) / 3)
    cand = got_links[None] * z[:, None, None, None]
    err = np.abs(cand - want_links[None]).reshape(3, len(got_links), -1).max(axis=2)
    best = err.argmin(axis=0)
    fixed = cand[best, np.arange(len(got_links))]
    return fixed, int((best != 0).sum())
