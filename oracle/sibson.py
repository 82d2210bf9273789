"""Sibson natural-neighbour weights by half-plane clipping (oracle; see oracle/__init__.py).

Definition (Sibson 1981, cited PAPER.md:153-157, eq. 8).  Let V_P(p) be the Voronoi cell of parent p among the
parents P, and C(x) the Voronoi cell the query point x would own in P + {x}.  Then

    w_p(x) = area(C(x) & V_P(p)) / area(C(x)),     w_p >= 0,   sum_p w_p = 1,

nonzero only for the parents whose cells x would steal from ("parents surrounding h_b").  Each Voronoi cell is
an intersection of half-planes {y : |y - a| <= |y - b|}; this file forms those intersections literally, by
clipping a convex polygon with one bisector at a time until no bisector cuts it any more.

SURVEY c8: coordinates are physical q = (hy/ly, hx/lx); all cells are clipped to the square |q_y|,|q_x| <=
2^10 qmax so that beams outside the parents' convex hull have a (far-field) definition; a beam coincident with
a parent gets the delta; weights < 1e-12 are dropped and the row renormalised.
"""
import numpy as np

DROP_BELOW = 1e-12
BOX_FACTOR = 1024.0


def _area(poly):
    """Shoelace area of a polygon given as [n, 2] vertices in order."""
    if poly.shape[0] < 3:
        return 0.0
    y, x = poly[:, 0], poly[:, 1]
    return 0.5 * abs(float(np.sum(x * np.roll(y, -1) - y * np.roll(x, -1))))


def _clip(poly, nrm, c):
    """Keep the part of the convex polygon with nrm . y <= c (one Sutherland-Hodgman step)."""
    if poly.shape[0] == 0:
        return poly
    s = poly @ nrm - c
    out = []
    n = poly.shape[0]
    for i in range(n):
        j = (i + 1) % n
        if s[i] <= 0.0:
            out.append(poly[i])
        if (s[i] < 0.0 < s[j]) or (s[j] < 0.0 < s[i]):
            t = s[i] / (s[i] - s[j])
            out.append(poly[i] + t * (poly[j] - poly[i]))
    return np.asarray(out, dtype=np.float64).reshape(-1, 2)


def _cell(poly, site, others, tol):
    """Intersect ``poly`` with the half-planes {y : |y - site| <= |y - o|} for every o in ``others``.
    |y-site|^2 <= |y-o|^2  <=>  2 (o - site) . y <= |o|^2 - |site|^2.
    Returns the polygon and the list of indices into ``others`` whose bisector actually cut it."""
    nrm = 2.0 * (others - site[None, :])
    c = np.sum(others * others, axis=1) - float(site @ site)
    used = np.zeros(others.shape[0], dtype=bool)
    cutters = []
    while poly.shape[0] >= 3:
        viol = (poly @ nrm.T - c[None, :]).max(axis=0)     # worst vertex per half-plane
        viol[used] = -np.inf
        k = int(np.argmax(viol))
        if viol[k] <= tol:
            break
        used[k] = True
        cutters.append(k)
        poly = _clip(poly, nrm[k], c[k])
    return poly, cutters


def sibson_row(x, parents_q, qmax, prune=True):
    """Weights of one query point x (physical q, shape [2]) on the parents ([P, 2]).
    Returns (indices ascending, weights).

    prune: work on the nearest parents only, when that provably changes nothing.  Let R be the largest distance
    from x to a vertex of C(x).  A parent o with |o - x| > 2R cannot bound C(x) (every y in C(x) has
    |y - o| >= |o - x| - R > R >= |y - x|), and a parent o with |o - x| > 4R cannot bound C(x) & V_P(p) for a
    neighbour p (|y - p| <= |y - x| + |x - p| <= 3R < |o - x| - R <= |y - o|).  So the cell is first built from
    the k nearest parents and accepted if every other parent is farther than 4R; otherwise k is doubled."""
    parents_q = np.asarray(parents_q, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    hit = np.nonzero(np.all(parents_q == x[None, :], axis=1))[0]
    if hit.size:
        return hit[:1].astype(np.int64), np.ones(1)
    if prune and parents_q.shape[0] > 64:
        d2 = np.sum((parents_q - x[None, :]) ** 2, axis=1)
        order = np.argsort(d2, kind="stable")
        k = 48
        while k < parents_q.shape[0]:
            near = order[:k]
            half = BOX_FACTOR * qmax
            box = np.array([[-half, -half], [-half, half], [half, half], [half, -half]], dtype=np.float64)
            cx, _ = _cell(box, x, parents_q[near], 1e-13 * half * half)
            R2 = np.max(np.sum((cx - x[None, :]) ** 2, axis=1))
            if d2[order[k]] > 16.0 * R2:                       # every excluded parent is farther than 4R
                idx, w = sibson_row(x, parents_q[near], qmax, prune=False)
                idx = near[idx]
                o = np.argsort(idx)
                return idx[o].astype(np.int64), w[o]
            k *= 2
    half = BOX_FACTOR * qmax
    box = np.array([[-half, -half], [-half, half], [half, half], [half, -half]], dtype=np.float64)
    tol = 1e-13 * half * half
    cx, cutters = _cell(box, x, parents_q, tol)             # C(x)
    total = _area(cx)
    idx, w = [], []
    for p in cutters:                                       # only a parent whose bisector bounds C(x) can lose area
        others = np.delete(parents_q, p, axis=0)
        stolen, _ = _cell(cx, parents_q[p], others, tol)    # C(x) & V_P(p)
        a = _area(stolen) / total
        if a >= DROP_BELOW:
            idx.append(p)
            w.append(a)
    idx = np.asarray(idx, dtype=np.int64)
    w = np.asarray(w, dtype=np.float64)
    order = np.argsort(idx)
    idx, w = idx[order], w[order]
    return idx, w / w.sum()


def natural_neighbour_weights(beams, parent_pos, ly, lx, qmax, rows=None):
    """Weight table of every beam (or of the listed ``rows``) on the parents (eq. 8).  ``parent_pos`` are positions
    of the parents inside ``beams``.  Returns a list of (indices into parents, weights) per requested row."""
    q = np.stack([beams[:, 0] / ly, beams[:, 1] / lx], axis=1)
    pq = q[parent_pos]
    rows = range(beams.shape[0]) if rows is None else rows
    return [sibson_row(q[b], pq, qmax) for b in rows]


def to_dense(table, n_parents):
    """[(idx, w)] -> dense [n_rows, n_parents] float64."""
    W = np.zeros((len(table), n_parents))
    for b, (idx, w) in enumerate(table):
        W[b, idx] = w
    return W
