"""Helpers shared by the tests (host side only)."""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def paper_values():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = [s.strip() for s in line.split("=")]
            out[k] = float(v)
    return out


J6 = np.zeros((6, 6))
for _i in range(3):
    J6[2 * _i, 2 * _i + 1] = 1.0
    J6[2 * _i + 1, 2 * _i] = -1.0


def unit_bunch(scale=1.0):
    """7 particles: the origin and the 6 unit vectors times `scale` -> columns of a linear map."""
    c = [np.zeros(7) for _ in range(6)]
    for j in range(6):
        c[j][j + 1] = scale
    return c


def matrix_of(track_fn, scale=1.0):
    """6x6 matrix of a LINEAR map given as track_fn(coords) (in place)."""
    c = unit_bunch(scale)
    track_fn(c)
    M = np.array([[c[i][j + 1] - c[i][0] for j in range(6)] for i in range(6)]) / scale
    assert all(c[i][0] == 0.0 for i in range(6)), "linear map must fix the origin"
    return M


def rms_emittance(q, p):
    q = q - q.mean()
    p = p - p.mean()
    return np.sqrt((q * q).mean() * (p * p).mean() - (q * p).mean() ** 2)


def r14_error(got, ref):
    """SURVEY R14 metric: max over particles of |got-ref| / max(|ref|, rms(ref)), per coordinate."""
    errs = []
    for g, r in zip(got, ref):
        rms = np.sqrt(np.mean(r * r))
        den = np.maximum(np.abs(r), rms)
        den = np.where(den > 0, den, 1.0)
        errs.append(float(np.max(np.abs(g - r) / den)) if r.size else 0.0)
    return errs
