"""Pin for the oracle's spawn keying (reading G11; oracle/philox.cpp child_id, used by oracle/track.cpp when a
scattering event creates a superphoton; north_star: "counter-based RNG keyed per superphoton").

G11: the id of the superphoton spawned by event j of a parent is the first 96 bits of
    Philox4x32-10(counter = (parent.i0, parent.i1, parent.i2, j), key = (seed_lo ^ TAG_SPAWN, seed_hi)),
and every later draw of that superphoton (TAG_STEP, TAG_SCAT streams) is keyed by this id.  A mistake here -- j not mixed
in, a parent word left out, a truncated id -- gives siblings (or cousins) the same or colliding random streams: that
inflates the variance without biasing any mean, so none of the physics pins can see it.  What pins it here:

  1. the ids equal the block of a Philox written a second time in this file (vectorised numpy on uint64), which is itself
     held to the three known-answer vectors of tests/golden/philox_kat.txt;
  2. over > 1e6 (parent, j) pairs shaped like a real config-1 run (every primary of the run, the event ordinals the
     oracle's own histories reach, and a second generation whose parents are 96-bit child ids), no two children share an
     id and none has the id of a primary (i2 == 0, (i1, i0) < number of primaries);
  3. the first TAG_STEP uniforms of siblings j and j+1 are uncorrelated (chi^2 of the 16 x 16 contingency table), and so
     are those of the children (same j) of consecutive primaries.

Perturbations tried on oracle/philox.cpp before committing (each makes this file fail): counter word 3 = 0 instead of j
(1, 2 and 3 fail: siblings get one id); counter word 2 = 0 instead of parent.i2 (1 fails on the second generation);
returned i2 forced to 0 (1 fails; 2 fails: such an id can be a primary's and the second generation collides in 64 bits
only by chance, but the primary-id check is deterministic for small i0,i1 -- see the assertion on i2).
"""
import os

import numpy as np

import paper_2602_13198_b200.workloads as wl
from oracle_binding import Oracle

HERE = os.path.dirname(__file__)
TAG_STEP, TAG_SPAWN = 0x53544550, 0x5350574E        # "STEP", "SPWN" (oracle/oracle.hpp enum Tag)
M0, M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
W0, W1 = 0x9E3779B9, 0xBB67AE85
MASK = np.uint64(0xFFFFFFFF)
S32 = np.uint64(32)


def philox_np(ctr, key):
    """Philox4x32-10 on arrays: ctr [n][4], key [2] or [n][2] (uint32 values held in uint64) -> [n][4]."""
    c = [np.asarray(ctr)[:, i].astype(np.uint64) for i in range(4)]
    key = np.asarray(key, dtype=np.uint64)
    k0, k1 = (key[..., 0] & MASK), (key[..., 1] & MASK)
    for _ in range(10):
        p0, p1 = M0 * c[0], M1 * c[2]                   # 32 x 32 -> 64 bits: exact in uint64
        c = [(p1 >> S32) ^ c[1] ^ k0, p1 & MASK, (p0 >> S32) ^ c[3] ^ k1, p0 & MASK]
        k0, k1 = (k0 + np.uint64(W0)) & MASK, (k1 + np.uint64(W1)) & MASK
    return np.stack(c, axis=1)


def unit_np(hi, lo):
    return (((hi << S32) | lo) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def test_the_second_philox_meets_the_known_answers():
    n = 0
    for line in open(os.path.join(HERE, "golden", "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        assert philox_np(np.array([w[0:4]]), np.array(w[4:6]))[0].tolist() == w[6:10]
        n += 1
    assert n == 3


def _pairs_like_config1(olib):
    """(seed, number of primaries, parents [n][3], j [n]) covering what a config-1 run at N_s = 1e6 asks of child_id."""
    p, prim = wl.config1(Ns=1e6)
    o = Oracle(p, prim)
    n_prim = o.prepare()
    tr, _, _ = o.trace(np.arange(0, n_prim, max(1, n_prim // 1500))[:1500])     # real histories: how many events a parent has
    jmax = int(tr["jscat"].max())
    assert jmax >= 2, "config 1 is the scattering sphere: its primaries scatter more than once"
    nj = max(jmax + 1, 4)
    pid = np.arange(n_prim, dtype=np.uint64)
    gen0 = np.stack([pid & MASK, pid >> S32, np.zeros_like(pid)], axis=1)       # primaries: (lo, hi, 0) (oracle/emit.cpp)
    parents = np.repeat(gen0, nj, axis=0)
    j = np.tile(np.arange(nj, dtype=np.uint64), n_prim)
    seed = int(p["seed"])
    # second generation: children of the first 100,000 children, 4 events each
    c1 = olib.child_ids(seed, parents[:100_000], j[:100_000]).astype(np.uint64)
    parents = np.concatenate([parents, np.repeat(c1, 4, axis=0)])
    j = np.concatenate([j, np.tile(np.arange(4, dtype=np.uint64), len(c1))])
    return seed, n_prim, parents, j


def test_child_ids_are_the_spawn_block_distinct_and_never_a_primary(olib):
    seed, n_prim, parents, j = _pairs_like_config1(olib)
    assert len(j) >= 1_000_000
    got = olib.child_ids(seed, parents, j).astype(np.uint64)
    # 1. the definition, typed out: counter (i0, i1, i2, j), key (seed_lo ^ TAG_SPAWN, seed_hi), first three words
    ctr = np.concatenate([parents, j[:, None]], axis=1)
    blk = philox_np(ctr, np.array([(seed & 0xFFFFFFFF) ^ TAG_SPAWN, seed >> 32]))
    assert np.array_equal(got, blk[:, :3])
    # 2. distinct in all 96 bits (as two keys: (i2, i1) and i0), and in particular between siblings
    hi = (got[:, 2] << S32) | got[:, 1]
    rows = np.stack([hi, got[:, 0]], axis=1)
    assert len(np.unique(rows, axis=0)) == len(rows)
    sib = got.reshape(-1, 3)[: (len(got) // 2) * 2].reshape(-1, 2, 3)           # (j, j+1) of one parent (nj is even or the
    assert np.all(np.any(sib[:, 0] != sib[:, 1], axis=1))                       #  pair spans two parents: still distinct)
    # a primary's id is (lo, hi, 0) with hi:lo < n_prim; a child id with i2 == 0 happens with probability 2^-32 per child
    as_primary = (got[:, 2] == 0) & (((got[:, 1] << S32) | got[:, 0]) < np.uint64(n_prim))
    assert not as_primary.any()
    assert np.count_nonzero(got[:, 2]) >= len(got) - 2                          # the third word is in use (truncated ids fail)
    # all three words carry entropy: each bit of each word is set in about half the ids
    for w in range(3):
        for b in (0, 7, 15, 16, 24, 31):
            f = np.mean((got[:, w] >> np.uint64(b)) & np.uint64(1))
            assert abs(f - 0.5) < 5 * 0.5 / np.sqrt(len(got)), (w, b, f)


def _chi2_independence(u, v, nb=16):
    h, _, _ = np.histogram2d(u, v, bins=nb, range=[[0, 1], [0, 1]])
    e = np.outer(h.sum(1), h.sum(0)) / h.sum()
    return float(((h - e) ** 2 / e).sum())


def test_streams_of_siblings_and_of_neighbouring_parents_are_uncorrelated(olib):
    seed, n_prim, parents, j = _pairs_like_config1(olib)
    n = 400_000
    ids = olib.child_ids(seed, parents[:n], j[:n]).astype(np.uint64)
    key = np.array([(seed & 0xFFFFFFFF) ^ TAG_STEP, seed >> 32])
    blk = philox_np(np.concatenate([ids, np.zeros((n, 1), dtype=np.uint64)], axis=1), key)     # step 0 of each child
    ux, ur = unit_np(blk[:, 0], blk[:, 1]), unit_np(blk[:, 2], blk[:, 3])
    # (the same numbers the oracle's tracker draws: oracle/track.cpp uniform_pair(seed, TAG_STEP, id, nstep))
    for i in (0, 1, 77777, n - 1):
        s = olib.stream(seed, TAG_STEP, int(ids[i, 0]), int(ids[i, 1]), int(ids[i, 2]), 2)
        assert s[0] == ux[i] and s[1] == ur[i]
    nj = int(j[: n].max()) + 1
    first = np.arange(0, n - 1)
    same_parent = (first % nj) != nj - 1
    a, b = first[same_parent], first[same_parent] + 1                           # siblings j, j+1
    dof = 15 * 15
    for u, v in ((ux[a], ux[b]), (ur[a], ur[b]), (ux[a], ur[b])):
        c2 = _chi2_independence(u, v)
        assert abs(c2 - dof) < 5 * np.sqrt(2 * dof), c2                         # 225 +- 5 sigma (sigma = 21.2)
        assert abs(np.corrcoef(u, v)[0, 1]) < 5 / np.sqrt(len(u))
    # children with the same j of consecutive primaries
    a = np.arange(0, n - nj)
    c2 = _chi2_independence(ux[a], ux[a + nj])
    assert abs(c2 - dof) < 5 * np.sqrt(2 * dof), c2
    # and each stream by itself is uniform
    h, _ = np.histogram(ux, bins=256, range=(0, 1))
    chi = float(((h - n / 256) ** 2 / (n / 256)).sum())
    assert abs(chi - 255) < 5 * np.sqrt(2 * 255), chi
