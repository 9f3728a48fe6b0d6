"""Seeded explicit frame lists for the frame-list mode.

The paper challenges the pairs that survive the exhaustive five-world prefix on named templates of
six to sixteen worlds ("paths, reverse paths, looped paths, and forked paths"; "path,
reverse-path, reflexive-path, fork, cycle, star, sparse, and dense templates at each size from six
through sixteen") and on synthesized relations ("stratified Erdos-Renyi sampling,
edge-flip mutation of canonical seeds, ... dead-end insertion, back-edge injection").
Its template list and generator parameters are not published; the families below take their shape
and stand in for them.

This module holds no evaluation: it only produces relations.  A frame list is a numpy array
`rel` of shape (F, n, n), dtype uint8, rel[j, w, u] = 1 iff frame j has the edge w -> u.  Both the
oracle (which reads the matrices as they are) and the CUDA path (which takes successor masks,
`succ_masks`) are fed from the same arrays.
"""
from __future__ import annotations

import numpy as np

SEED_FRAMES = 15437006


def _empty(n):
    return np.zeros((n, n), np.uint8)


def path(n):
    """0 -> 1 -> ... -> n-1 (the frame of Proposition 5 for n = 6)."""
    r = _empty(n)
    for w in range(n - 1):
        r[w, w + 1] = 1
    return r


def reverse_path(n):
    return path(n).T.copy()


def reflexive_path(n):
    r = path(n)
    for w in range(n):
        r[w, w] = 1
    return r


def fork(n):
    """A path 0 -> ... -> n-3 whose end branches to the two leaves n-2 and n-1."""
    r = _empty(n)
    if n < 3:
        return path(n)
    for w in range(n - 3):
        r[w, w + 1] = 1
    r[n - 3, n - 2] = 1
    r[n - 3, n - 1] = 1
    return r


def cycle(n):
    r = path(n)
    r[n - 1, 0] = 1
    return r


def star(n):
    r = _empty(n)
    r[0, 1:] = 1
    return r


def reverse_star(n):
    return star(n).T.copy()


def path_with_loop_end(n):
    """A path whose last world sees itself (no dead end)."""
    r = path(n)
    r[n - 1, n - 1] = 1
    return r


def complete(n):
    return np.ones((n, n), np.uint8)


def empty(n):
    return _empty(n)


TEMPLATES = {
    "path": path, "reverse_path": reverse_path, "reflexive_path": reflexive_path, "fork": fork,
    "cycle": cycle, "star": star, "reverse_star": reverse_star, "path_loop_end": path_with_loop_end,
    "complete": complete, "empty": empty,
}


def templates(n):
    """Every named template at size n, in the fixed order of TEMPLATES: (names, rel[F, n, n])."""
    names = list(TEMPLATES)
    return names, np.stack([TEMPLATES[t](n) for t in names])


def erdos_renyi(n, count, seed=SEED_FRAMES, densities=(0.05, 0.1, 0.2, 0.35, 0.5, 0.8)):
    """Stratified Erdos-Renyi relations: frame j uses density densities[j % len(densities)]; every
    ordered pair (including loops) is an edge independently with that probability."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000003 * n))
    p = np.asarray(densities, np.float64)[np.arange(count) % len(densities)]
    u = rng.random((count, n, n))
    return (u < p[:, None, None]).astype(np.uint8)


def edge_flip(n, count, seed=SEED_FRAMES, max_flips=4):
    """Edge-flip mutation of canonical seeds: frame j starts from template j % len(TEMPLATES) and
    has 1..max_flips uniformly chosen ordered pairs toggled."""
    rng = np.random.Generator(np.random.PCG64(seed + 7 + 1000003 * n))
    _, base = templates(n)
    rel = base[np.arange(count) % len(base)].copy()
    flips = rng.integers(1, max_flips + 1, size=count)
    pos = rng.integers(0, n * n, size=(count, max_flips))
    flat = rel.reshape(count, n * n)
    for t in range(max_flips):
        on = flips > t
        idx = np.nonzero(on)[0]
        flat[idx, pos[idx, t]] ^= 1
    return rel


def dead_end_insertion(n, count, seed=SEED_FRAMES, density=0.3):
    """Erdos-Renyi relations in which one seeded world is made a dead end (its row cleared)."""
    rng = np.random.Generator(np.random.PCG64(seed + 13 + 1000003 * n))
    rel = (rng.random((count, n, n)) < density).astype(np.uint8)
    dead = rng.integers(0, n, size=count)
    rel[np.arange(count), dead, :] = 0
    return rel


def back_edge_injection(n, count, seed=SEED_FRAMES):
    """The path 0 -> ... -> n-1 plus one or two seeded back edges w -> u with u <= w."""
    rng = np.random.Generator(np.random.PCG64(seed + 29 + 1000003 * n))
    rel = np.repeat(path(n)[None], count, axis=0)
    for _ in range(2):
        w = rng.integers(0, n, size=count)
        u = (rng.random(count) * (w + 1)).astype(np.int64)
        rel[np.arange(count), w, u] = 1
    return rel


def stress_list(n, count, seed=SEED_FRAMES):
    """The mixed list used by tests and bench.py: the templates, then Erdos-Renyi, edge-flip,
    dead-end and back-edge relations in equal shares, `count` frames in total."""
    _, t = templates(n)
    rest = max(0, count - len(t))
    q = [rest // 4 + (1 if i < rest % 4 else 0) for i in range(4)]
    parts = [t[:count], erdos_renyi(n, q[0], seed), edge_flip(n, q[1], seed),
             dead_end_insertion(n, q[2], seed), back_edge_injection(n, q[3], seed)]
    return np.concatenate([p for p in parts if len(p)], axis=0)


def succ_masks(rel):
    """rel[F, n, n] -> successor masks uint16[F, n]: bit u of succ[j, w] is the edge w -> u (the
    input format of kripke_eval_frames; a change of representation, no evaluation)."""
    F, n, _ = rel.shape
    weights = (1 << np.arange(n, dtype=np.uint32)).astype(np.uint32)
    return (rel.astype(np.uint32) * weights[None, None, :]).sum(axis=2).astype(np.uint16)
