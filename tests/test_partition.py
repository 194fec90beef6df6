"""Host logic of the fused step kernels' work partition, through the C ABI's
host-only fdtd_debug_partition: no GPU needed.  Checked against what the partition must guarantee, not
against its own arithmetic: every (tile, plane) position is marched exactly once, runs have (almost) equal
model cost, and in the lock-step split y-adjacent columns of one cost class have identical cuts."""
import collections

import pytest


def _b():
    from paper_2412_12360_b200 import build
    build.build()
    from paper_2412_12360_b200 import binding
    return binding


def _cost(j0, k, ny, nz, d, ty, wy, wz):
    ys = d > 0 and (j0 <= d or j0 + ty >= ny - d)
    zs = d > 0 and (k <= d or k >= nz - d - 1)
    return 1.0 + (wy if ys else 0.0) + (wz if zs else 0.0)


CASES = [
    # nx, ny, nz, d, tile_x, tile_y, n_cta
    (200, 200, 200, 12, 200, 7, 148),      # C3 in the bench configuration
    (88, 52, 44, 6, 64, 7, 37),            # ragged tails in x and y, two tile columns in x
    (800, 800, 600, 16, 200, 7, 148),      # C4
    (64, 64, 64, 10, 64, 7, 148),          # C2: fewer planes per run than CPML cells
    (16, 16, 16, 0, 16, 3, 5),             # no CPML: one cost class
]


@pytest.mark.parametrize("lockstep", [True, False])
@pytest.mark.parametrize("case", CASES)
def test_every_position_exactly_once_and_costs_balanced(case, lockstep):
    b = _b()
    nx, ny, nz, d, tx, ty, n_cta = case
    wy, wz = 1.0, 0.8
    segs = b.fdtd_debug_partition(nx, ny, nz, d, tx, ty, n_cta, wy, wz, lockstep)
    seen = collections.Counter()
    cost = collections.defaultdict(float)
    ctas = []
    for cta, i0, j0, k0, k1 in segs:
        assert 0 <= cta < n_cta and i0 % tx == 0 and j0 % ty == 0 and 0 <= i0 < nx and 0 <= j0 < ny
        assert 0 <= k0 < k1 <= nz
        if not ctas or ctas[-1] != cta:
            ctas.append(cta)
        for k in range(k0, k1):
            seen[(i0, j0, k)] += 1
            cost[cta] += _cost(j0, k, ny, nz, d, ty, wy, wz)
    assert ctas == list(range(n_cta))                       # every CTA has work, segments grouped by CTA
    n_cols = -(-nx // tx) * -(-ny // ty)
    assert len(seen) == n_cols * nz and set(seen.values()) == {1}
    mean = sum(cost.values()) / n_cta
    worst_plane = 1.0 + wy + wz
    assert max(cost.values()) <= mean + 2 * worst_plane     # cuts fall on plane boundaries: at most ~a plane off per side
    assert min(cost.values()) >= mean - 2 * worst_plane


def test_lockstep_columns_of_one_class_share_their_cuts():
    b = _b()
    nx = ny = nz = 200
    d, tx, ty, n_cta = 12, 200, 7, 148
    segs = b.fdtd_debug_partition(nx, ny, nz, d, tx, ty, n_cta, 1.0, 0.8, True)
    per_cta = collections.defaultdict(list)
    for s in segs:
        per_cta[s[0]].append(s)
    # full runs = CTAs with one segment; their cuts per column
    cuts = collections.defaultdict(set)
    single = 0
    for cta, ss in per_cta.items():
        if len(ss) == 1:
            single += 1
            _, i0, j0, k0, k1 = ss[0]
            cuts[j0].update((k0, k1))
    interior = [j0 for j0 in range(0, ny, ty) if not (j0 <= d or j0 + ty >= ny - d) and j0 + ty <= ny]
    assert len(interior) >= 20
    ref = cuts[interior[0]]
    assert len(ref) >= 4                                    # several full runs per interior column
    for j0 in interior:
        assert cuts[j0] == ref                              # identical cuts: the columns march in lock step
    assert single >= 0.85 * n_cta                           # what is chained from the column tops is a small remainder
    # the plain split does not have this property (that is what the lock-step split fixes)
    plain = b.fdtd_debug_partition(nx, ny, nz, d, tx, ty, n_cta, 1.0, 0.8, False)
    starts = collections.defaultdict(set)
    for cta, i0, j0, k0, k1 in plain:
        starts[j0].add(k0)
    assert starts[interior[0]] != starts[interior[1]]


def test_bad_arguments_are_rejected():
    b = _b()
    with pytest.raises(b.FdtdError):
        b.fdtd_debug_partition(0, 8, 8, 0, 8, 3, 2)
    with pytest.raises(b.FdtdError):
        b.fdtd_debug_partition(8, 8, 8, 0, 8, 8, 100)       # more CTAs than positions


def test_large_grids_march_whole_columns_in_waves():
    """More columns than CTAs (C4): the columns without a y slab are dealt out whole, in sequence order, CTA c taking
    the c-th, (c + n_cta)-th, ... of them, so the n_cta y-consecutive columns of a wave start at plane 0 together;
    only the other columns (the pool that levels the costs) are cut inside."""
    b = _b()
    nx, ny, nz, d, tx, ty, n_cta = 800, 800, 600, 16, 200, 7, 148
    nty = -(-ny // ty)
    segs = b.fdtd_debug_partition(nx, ny, nz, d, tx, ty, n_cta, 1.0, 0.8, True)
    col = lambda s: (s[0] // tx) * nty + s[1] // ty
    slab = lambda j0: j0 <= d or j0 + ty >= ny - d
    cheap = [t for t in range(4 * nty) if not slab((t % nty) * ty)]
    per_cta = collections.defaultdict(list)
    for s in segs:
        per_cta[s[0]].append(s[1:])
    whole = 0
    for c in range(n_cta):
        w = 0
        while w < len(per_cta[c]) and per_cta[c][w][2:] == (0, nz):
            assert col(per_cta[c][w]) == cheap[c + w * n_cta]
            w += 1
        assert w >= 2
        whole += w
        for s in per_cta[c][w:]:                              # what follows is pool work: columns with a y slab
            assert slab(s[1])
    assert whole == len(cheap)                                # every cheap column is marched whole: 440 of 460
