"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ and workloads/.

    python tests/golden/make_golden.py <part> [--threads N]

parts (sizes are oracle evaluations; times are for the 8-core build box at ~0.1 G eval/s):
  c2          config 2: 5,624 formulas, n=4, classes K/T/S4/S5, full ranges      (1.0e11, ~15 min)
  n5_classes  config 3: same corpus, n=5, classes S4 and S5 in full             (4.0e10, ~6 min)
  n5_ranges   config 3: 16 seeded ranges of 2^10 frames of K and of T at n=5, every formula
              (SURVEY 8(c) plan item 4; 1.9e11, ~25 min)
  n5_orbit    config 3: full-range K counts at n=5 for 200 seeded NON-CONSTANT corpus formulas (at
              least 100 of them over both variables) and the named axioms, by the isomorphism-orbit
              route (291,968 representatives x orbit sizes; plan item 5)
  n5_t_full   config 3: 120 seeded non-constant corpus formulas over ALL 2^20 reflexive frames at
              n=5 (plan item 3; 1.3e11, ~15 min)
  c4_ranges   config 4: 2,048 three-variable formulas, n=5, 4 seeded ranges of 8 K-frames
  c5_counts   config 5: distinguishing-frame counts of every pair for n=1..5 (orbit route at
              n=5) and first witnesses for n<=4

  c3_paper    the paper-shaped census corpus: the 44,678 constant-free formulas of <= 7 nodes over
              {p, q}, one representative (first in enumeration order) per class of equal truth sets on all
              models of <= 3 worlds (oracle signatures: 5,621) + the K axiom; at n=5: S4 and S5 in full,
              8 seeded ranges of 2^10 frames of K and of T for every formula, and full-range K counts of
              100 seeded two-variable representatives by the orbit route (1.7e11, ~25 min)

Nothing here imports the CUDA path; no value comes from it.  Each .npz stores the corpus SHA-256
so a test can tell that it is comparing the same bytes.
"""
import argparse
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import workloads as W                      # noqa: E402
from oracle import volume as V             # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
CLASSES = {"K": 0, "T": 1, "S4": 2, "S5": 3}


def sha(programs):
    return hashlib.sha256(b"\xff".join(programs)).hexdigest()


def seeded_ranges(seed, total, width, count):
    rng = W.SplitMix64(seed)
    return sorted(rng.below(total - width) for _ in range(count))


def save(name, **arrays):
    path = os.path.join(HERE, name)
    np.savez_compressed(path, **arrays)
    print("wrote", path, os.path.getsize(path), "bytes")


def part_c2(threads):
    progs = W.corpus_c2()
    code, offs = W.pack_programs(progs)
    out = {"corpus_sha256": np.array(sha(progs))}
    for cname, cls in CLASSES.items():
        t = time.time()
        r = V.census(code, offs, 4, 2, cls, threads=threads)
        print(cname, "%.1fs" % (time.time() - t))
        for key, val in r.items():
            out[f"{cname}_{key}"] = val
    save("c2_n4.npz", **out)


def part_n5_classes(threads):
    progs = W.corpus_c2()
    code, offs = W.pack_programs(progs)
    out = {"corpus_sha256": np.array(sha(progs))}
    for cname in ("S4", "S5"):
        t = time.time()
        r = V.census(code, offs, 5, 2, CLASSES[cname], threads=threads)
        print(cname, "%.1fs" % (time.time() - t))
        for key, val in r.items():
            out[f"{cname}_{key}"] = val
    save("n5_s4s5.npz", **out)


def seeded_formulas(seed, want, min_two_var=0):
    """Indices into corpus_c2(): `want` distinct non-constant formulas drawn by seed from the whole
    corpus ('non-constant' = mentions a variable), at least min_two_var of them over both p and q."""
    progs = W.corpus_c2()
    rng = W.SplitMix64(seed)
    two = [i for i, c in enumerate(progs) if b"\x10" in c and b"\x11" in c]
    some = [i for i, c in enumerate(progs) if b"\x10" in c or b"\x11" in c]
    picked = set()
    while len(picked) < min_two_var:
        picked.add(two[rng.below(len(two))])
    while len(picked) < want:
        picked.add(some[rng.below(len(some))])
    return sorted(picked)


def part_n5_ranges(threads):
    progs = W.corpus_c2()
    code, offs = W.pack_programs(progs)
    width = 1 << 10
    out = {"corpus_sha256": np.array(sha(progs)), "width": np.array(width)}
    for cname, total, seed in (("K", 1 << 25, 501), ("T", 1 << 20, 502)):
        begins = seeded_ranges(seed, total, width, 16)
        out[f"{cname}_begin"] = np.array(begins, np.uint64)
        acc = {}
        for b in begins:
            r = V.census(code, offs, 5, 2, CLASSES[cname], b, width, threads=threads)
            for key, val in r.items():
                acc.setdefault(key, []).append(val)
        for key, val in acc.items():
            out[f"{cname}_{key}"] = np.stack(val)
    save("n5_ranges.npz", **out)


def part_n5_t_full(threads):
    corpus = W.corpus_c2()
    idx = seeded_formulas(503, 120, 60)
    progs = [corpus[i] for i in idx]
    code, offs = W.pack_programs(progs)
    t = time.time()
    r = V.census(code, offs, 5, 2, CLASSES["T"], threads=threads)
    print("T full census %.1fs" % (time.time() - t))
    save("n5_t_full.npz", corpus_sha256=np.array(sha(progs)), index=np.array(idx, np.uint32), **r)


def part_n5_orbit(threads):
    corpus = W.corpus_c2()
    idx = seeded_formulas(505, 200, 100)
    progs = [corpus[i] for i in idx] + [W.to_postfix(t) for t in W.named_axioms().values()]
    code, offs = W.pack_programs(progs)
    reps, sizes = V.orbits(5)
    assert int(sizes.sum()) == 1 << 25
    t = time.time()
    r = V.census_list(code, offs, 5, 2, reps, weights=sizes, threads=threads)
    print("orbit census %.1fs" % (time.time() - t))
    save("n5_orbit.npz", corpus_sha256=np.array(sha(progs)), index=np.array(idx, np.uint32),
         models=r["models"], frames=r["frames"])


def paper_corpus():
    """(programs, indices of the representatives in W.enumerate_constant_free(7, 2) order): P:143's reduction
    done by the oracle's signatures; the K axiom is appended last (R19)."""
    forms = W.enumerate_constant_free(7, 2)
    progs = [W.to_postfix(t) for t in forms]
    a, b = V.signatures(*W.pack_programs(progs), 3, 2)
    first = {}
    for i, s in enumerate(zip(a.tolist(), b.tolist())):
        first.setdefault(s, i)
    reps = sorted(first.values())
    return [progs[i] for i in reps] + [W.to_postfix(W.named_axioms()["K"])], np.array(reps, np.uint32), len(progs)


def part_c3_paper(threads):
    progs, reps, n_enum = paper_corpus()
    print(f"{n_enum} enumerated -> {len(reps)} representatives + K axiom")
    code, offs = W.pack_programs(progs)
    out = {"corpus_sha256": np.array(sha(progs)), "rep_index": reps, "n_enumerated": np.array(n_enum)}
    for cname in ("S4", "S5"):
        t = time.time()
        r = V.census(code, offs, 5, 2, CLASSES[cname], threads=threads)
        print(cname, "%.1fs" % (time.time() - t))
        for key, val in r.items():
            out[f"{cname}_{key}"] = val
    width = 1 << 10
    out["width"] = np.array(width)
    for cname, total, seed in (("K", 1 << 25, 511), ("T", 1 << 20, 512)):
        begins = seeded_ranges(seed, total, width, 8)
        out[f"{cname}_begin"] = np.array(begins, np.uint64)
        acc = {}
        t = time.time()
        for b in begins:
            r = V.census(code, offs, 5, 2, CLASSES[cname], b, width, threads=threads)
            for key, val in r.items():
                acc.setdefault(key, []).append(val)
        print(cname, "ranges %.1fs" % (time.time() - t))
        for key, val in acc.items():
            out[f"{cname}_{key}"] = np.stack(val)
    # full-range K counts of 100 seeded representatives over both variables, by the orbit route
    rng = W.SplitMix64(513)
    two = [i for i, c in enumerate(progs) if b"\x10" in c and b"\x11" in c]
    picked = set()
    while len(picked) < 100:
        picked.add(two[rng.below(len(two))])
    idx = sorted(picked)
    oc, oo = W.pack_programs([progs[i] for i in idx])
    orb, sizes = V.orbits(5)
    assert int(sizes.sum()) == 1 << 25
    t = time.time()
    r = V.census_list(oc, oo, 5, 2, orb, weights=sizes, threads=threads)
    print("orbit census %.1fs" % (time.time() - t))
    out["orbit_index"] = np.array(idx, np.uint32)
    out["orbit_models"], out["orbit_frames"] = r["models"], r["frames"]
    save("c3_paper_n5.npz", **out)


def part_c4_ranges(threads):
    progs = W.corpus_c4()
    code, offs = W.pack_programs(progs)
    begins = seeded_ranges(504, 1 << 25, 8, 4)
    acc = {}
    for b in begins:
        r = V.census(code, offs, 5, 3, 0, b, 8, threads=threads)
        for key, val in r.items():
            acc.setdefault(key, []).append(val)
    save("c4_ranges.npz", corpus_sha256=np.array(sha(progs)), begin=np.array(begins, np.uint64),
         width=np.array(8), **{k: np.stack(v) for k, v in acc.items()})


def part_c5_counts(threads):
    progs, pairs, names = W.pairs_c5()
    code, offs = W.pack_programs(progs)
    pairs = np.array(pairs, np.uint32)
    out = {"corpus_sha256": np.array(sha(progs)), "n_pairs": np.array(len(pairs))}
    for n in (1, 2, 3, 4):
        r = V.census(code, offs, n, 0, 0, pairs=pairs, threads=threads)
        for key in ("frames", "wit_f", "wit_w"):
            out[f"n{n}_{key}"] = r[key]
    reps, sizes = V.orbits(5)
    r = V.census_list(code, offs, 5, 0, reps, weights=sizes, pairs=pairs, threads=threads)
    out["n5_frames"] = r["frames"]
    save("c5_counts.npz", **out)


PARTS = {"c2": part_c2, "n5_classes": part_n5_classes, "n5_ranges": part_n5_ranges,
         "n5_orbit": part_n5_orbit, "n5_t_full": part_n5_t_full, "c4_ranges": part_c4_ranges, "c5_counts": part_c5_counts,
         "c3_paper": part_c3_paper}

if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("part", choices=sorted(PARTS) + ["all"])
    ap.add_argument("--threads", type=int, default=0)
    a = ap.parse_args()
    V.build()
    for p in (sorted(PARTS) if a.part == "all" else [a.part]):
        t0 = time.time()
        PARTS[p](a.threads)
        print(p, "done in %.1fs" % (time.time() - t0))
