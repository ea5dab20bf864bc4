"""Oracle O1: grid arithmetic of 3D local-window clustering (test infrastructure).

Follows PAPER.md Alg. 2 lines 3-6 (l.352-356), lines 7-11 (l.357-363) and lines 15-18
(l.369-376); Eq. 5 (l.81).  The floor brackets are printed as |.| in PAPER.md (garbled);
they are floors (reading R-C4).

Pinned by: the paper's printed centroid counts 432 / 1215 / 336 / 960 and the 6.3x
search-space reduction (tests/golden/grid_counts.txt), brute-force window enumeration.
"""
from __future__ import annotations


def grid_dims(lattice, cell):
    """K_* = ceil(dim / k_*)   (Alg. 2 line 3, l.352)."""
    return tuple(-(-int(d) // int(k)) for d, k in zip(lattice, cell))


def clip_window(win, K):
    """w_* <- min(w_*, K_*)   (Alg. 2 line 4, l.353)."""
    return tuple(min(int(w), int(k)) for w, k in zip(win, K))


def window_start(u, w, K):
    """u_bar = clip(u - floor(w/2), 0, K - w)   (Alg. 2 lines 15-17, l.369-373)."""
    return min(max(u - w // 2, 0), K - w)


def centre_token(u, k, dim):
    """c = min(u*k + floor(k/2), dim-1)   (Alg. 2 lines 8-10, l.358-360)."""
    return min(u * k + k // 2, dim - 1)


def home_cell(coord, cell):
    """g(l) = (floor(t/k_t), floor(h/k_h), floor(w/k_w))   (Eq. 5, l.81)."""
    return tuple(c // k for c, k in zip(coord, cell))


def window_ids(u3, win, K):
    """N(u): linear ids of the clipped window of grid cell u3, enumerated delta_t-major,
    i.e. in ascending linear centroid id u = (u_t*K_h + u_h)*K_w + u_w
    (Alg. 2 line 18, l.375; tie-break reading R-C1)."""
    st = [window_start(u3[a], win[a], K[a]) for a in range(3)]
    ids = []
    for dt in range(win[0]):
        for dh in range(win[1]):
            for dw in range(win[2]):
                ids.append(((st[0] + dt) * K[1] + (st[1] + dh)) * K[2] + (st[2] + dw))
    return ids
