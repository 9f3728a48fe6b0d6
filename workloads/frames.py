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


# ---- counter-based generators: the numpy side of kripke_frames_generate (include/kripke.h) ----------------
# Frame j of a list depends only on (generator, n, seed, j): every draw is the SplitMix64 finaliser of a key.
# The library writes the same lists on the device (csrc/frame_gen.cu); tests compare the two element by
# element and feed the oracle from THIS side.  Input generation only: no formula is evaluated here.
GEN_TEMPLATES, GEN_ERDOS_RENYI, GEN_EDGE_FLIP, GEN_DEAD_END, GEN_BACK_EDGE, GEN_STRESS = range(6)
_DENSITY = np.array([214748364, 429496729, 858993459, 1503238553, 2147483648, 3435973836], np.uint64)  # x 2^-32
_DENSITY03 = np.uint64(1288490188)
_M = np.uint64


def _mix(x):
    with np.errstate(over="ignore"):
        x = (x + _M(0x9E3779B97F4A7C15)).astype(np.uint64)
        x = (x ^ (x >> _M(30))) * _M(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> _M(27))) * _M(0x94D049BB133111EB)
        return x ^ (x >> _M(31))


def _draw(seed, gen, n, j, t):
    """draw t of frame j (arrays broadcast)."""
    with np.errstate(over="ignore"):
        key = _mix(np.array(seed ^ (gen << 56) ^ (n << 48), np.uint64))
        return _mix(key + np.asarray(j, np.uint64) * _M(0xD6E8FEB86659FD93) + np.asarray(t, np.uint64) * _M(0x2545F4914F6CDD1D))


def generate_cb(gen, n, count, seed=SEED_FRAMES):
    """rel[count, n, n] of one counter-based generator (not GEN_STRESS)."""
    j = np.arange(count, dtype=np.uint64)
    names, base = templates(n)
    if gen == GEN_TEMPLATES:
        return base[(j % _M(len(base))).astype(np.int64)].copy()
    if gen in (GEN_ERDOS_RENYI, GEN_DEAD_END):
        t = np.arange(n * n, dtype=np.uint64)
        d = _draw(seed, gen, n, j[:, None], t[None, :]) >> _M(32)
        thr = _DENSITY[(j % _M(6)).astype(np.int64)][:, None] if gen == GEN_ERDOS_RENYI else _DENSITY03
        rel = (d < thr).astype(np.uint8).reshape(count, n, n)
        if gen == GEN_DEAD_END:
            dead = (_draw(seed, gen, n, j, 1000) % _M(n)).astype(np.int64)
            rel[np.arange(count), dead, :] = 0
        return rel
    if gen == GEN_EDGE_FLIP:
        rel = base[(j % _M(len(base))).astype(np.int64)].copy()
        flips = 1 + (_draw(seed, gen, n, j, 100) % _M(4)).astype(np.int64)
        flat = rel.reshape(count, n * n)
        for t in range(4):
            idx = np.nonzero(flips > t)[0]
            pos = (_draw(seed, gen, n, j[idx], t) % _M(n * n)).astype(np.int64)
            flat[idx, pos] ^= 1
        return rel
    if gen == GEN_BACK_EDGE:
        rel = np.repeat(path(n)[None], count, axis=0)
        for t in range(2):
            w = (_draw(seed, gen, n, j, 2 * t) % _M(n)).astype(np.int64)
            u = (_draw(seed, gen, n, j, 2 * t + 1) % (w + 1).astype(np.uint64)).astype(np.int64)
            rel[np.arange(count), w, u] = 1
        return rel
    raise ValueError(gen)


def stress_list_cb(n, count, seed=SEED_FRAMES):
    """The mixed list KRIPKE_GEN_STRESS writes: the templates, then the four generators in equal shares."""
    nt = min(count, len(TEMPLATES))
    rest = count - nt
    q = [rest // 4 + (1 if i < rest % 4 else 0) for i in range(4)]
    parts = [generate_cb(GEN_TEMPLATES, n, nt, seed)] + [generate_cb(GEN_ERDOS_RENYI + i, n, q[i], seed) for i in range(4)]
    return np.concatenate([p for p in parts if len(p)], axis=0)
