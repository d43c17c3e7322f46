"""Vectorised numpy restatement of the bin map, used ONLY by tests as an
independent cross-check of the oracle (numpy float32 arithmetic rounds every
operation once, no FMA).  Never imported by the oracle or the CUDA path."""
import numpy as np


def bins_f32(xy, cos_t, sin_t, rho_max, n_rho, scale=1):
    """[n_hits, n_theta] int32 bins, -1 where the vote is dropped."""
    xy = np.asarray(xy, dtype=np.float32)
    x, y = xy[:, 0], xy[:, 1]
    with np.errstate(all="ignore"):
        d = x * x + y * y
        u = np.float32(scale) * (x / d)
        v = np.float32(scale) * (y / d)
        rho = u[:, None] * cos_t[None, :] + v[:, None] * sin_t[None, :]
        inv = np.float32(np.float64(n_rho) / (2.0 * np.float64(np.float32(rho_max))))
        t = (rho + np.float32(rho_max)) * inv
        ok = (t >= 0) & (t < np.float32(n_rho))
        k = np.where(ok, np.where(ok, t, 0).astype(np.int32), -1)
    assert rho.dtype == np.float32 and t.dtype == np.float32
    return k


def bins_f64(xy, n_theta, rho_max, n_rho):
    """Same map in double precision with exact-as-possible theta (pin P6)."""
    xy = np.asarray(xy, dtype=np.float64)
    x, y = xy[:, 0], xy[:, 1]
    with np.errstate(all="ignore"):
        d = x * x + y * y
        u, v = x / d, y / d
        th = np.arange(n_theta) * (np.pi / n_theta)
        rho = u[:, None] * np.cos(th)[None, :] + v[:, None] * np.sin(th)[None, :]
        t = (rho + np.float64(np.float32(rho_max))) * (n_rho / (2.0 * np.float64(np.float32(rho_max))))
        ok = (t >= 0) & (t < n_rho)
        k = np.where(ok, np.floor(np.where(ok, t, 0)).astype(np.int64), -1)
    return k, t


def accumulate(bins, n_theta, n_rho):
    A = np.zeros((n_theta, n_rho), dtype=np.uint32)
    j = np.broadcast_to(np.arange(n_theta)[None, :], bins.shape)
    ok = bins >= 0
    np.add.at(A, (j[ok], bins[ok]), 1)
    return A


def dilate_peaks(peaks, n_theta, n_rho, w):
    """Boolean [n_theta, n_rho] union of the stored peaks' (theta, rho) windows."""
    D = np.zeros((n_theta, n_rho), dtype=bool)
    for j, k, _ in peaks:
        j, k = int(j), int(k)
        D[max(0, j - w):min(n_theta - 1, j + w) + 1, max(0, k - w):min(n_rho - 1, k + w) + 1] = True
    return D


def keep_from_dilation(bins, D):
    j = np.broadcast_to(np.arange(D.shape[0])[None, :], bins.shape)
    ok = bins >= 0
    hit = np.zeros(bins.shape, dtype=bool)
    hit[ok] = D[j[ok], bins[ok]]
    return hit.any(axis=1).astype(np.uint8)
