"""CPU checks of the integer identities the fast kernel's design rests on (hough_fast.cuh), modelled in numpy with the
kernel's word widths and compared with the oracle's definitions.  They do not run the kernel (the `-m gpu` parity tests
do); they pin the derivations stated in DESIGN.md section 7.1 at sizes the GPU tests cannot enumerate:

  * address folding: ((a' >> (F - k)) & ~(2^k - 1)) | column is the shared-memory address of the counter word,
    a' = u_q C + v_q S + O_q + (tile_base << (F - k)) in wrapping 32-bit arithmetic;
  * the threshold test on packed halfwords, (w + (2^15 - T) * 0x00010001) & 0x80008000;
  * the strict-local-maximum test of the 8 bins of a chunk on packed halfwords (column maxima, halfword shifts by byte
    permutation, borrow-free compares) == oracle O4 (`hough_def.peaks`);
  * the S3 join rules (prelinks inside a chunk, at most two explicit joins per on bin, implied joins skipped) connect
    exactly the 8-connected components (`scipy.ndimage.label`);
  * the Cauchy-Schwarz bounds behind the unchecked vote loop (safe radius) and the restricted clear / scan (reachable rows).
"""
import numpy as np
import pytest

from oracle import hough_def as D
from util import std_params

U32 = np.uint64(0xFFFFFFFF)


def _u32(x):
    return np.asarray(x, dtype=np.uint64) & U32


@pytest.mark.parametrize("n_theta,n_rho,G", [(512, 512, 2), (256, 256, 2), (256, 512, 1), (180, 256, 2), (128, 128, 1), (1024, 1024, 1)])
def test_vote_address_folding(n_theta, n_rho, G):
    """For every in-range (hit, theta) the folded 32-bit expression is tile_base + r * row_bytes + column, r = a >> F."""
    p = std_params(n_theta, n_rho)
    k = D.constants(p)
    row_bytes = 128 * G
    kk = int(np.log2(row_bytes))
    sh = k.F - kk
    assert sh >= 0
    tile_base = 1024  # dynamic shared memory window offset: a multiple of the row size, below 4096 (the kernel checks both at entry)
    assert ((4096 << sh) + (n_rho << k.F)) <= 0xFFFFFFFF  # the plan's admission test for the fast path
    rng = np.random.default_rng(7)
    lim = int(p.coord_max * (1 << k.H))
    uq = rng.integers(-lim, lim + 1, 4000)
    vq = rng.integers(-lim, lim + 1, 4000)
    C = np.asarray(k.Cq, dtype=np.int64)
    S = np.asarray(k.Sq, dtype=np.int64)
    a = uq[:, None] * C[None, :] + vq[:, None] * S[None, :] + k.Oq  # exact
    r = a >> k.F
    inr = (r >= 0) & (r < n_rho)
    assert inr.any()
    Oq2 = (k.Oq + (tile_base << sh)) & 0xFFFFFFFF
    a32 = _u32(_u32(uq[:, None] * C[None, :]) + _u32(_u32(vq[:, None] * S[None, :]) + np.uint64(Oq2)))  # wrapping IMADs
    amask = np.uint64((~((1 << kk) - 1)) & 0xFFFFFFFF)
    col = np.uint64(4 * 13)  # any lane's column offset inside the row (< row_bytes, word aligned)
    addr = ((a32 >> np.uint64(sh)) & amask) | col
    want = tile_base + r * row_bytes + int(col)
    np.testing.assert_array_equal(addr[inr].astype(np.int64), want[inr])


@pytest.mark.parametrize("T", [1, 19, 20, 24, 1023])
def test_packed_threshold_test(T):
    rng = np.random.default_rng(T)
    lo = rng.integers(0, 1 << 15, 20000, dtype=np.uint64)
    hi = rng.integers(0, 1 << 15, 20000, dtype=np.uint64)
    for near in (T - 1, T, T + 1):  # make sure the boundary is hit
        lo[rng.integers(0, lo.size, 500)] = max(near, 0)
        hi[rng.integers(0, hi.size, 500)] = max(near, 0)
    w = lo | (hi << np.uint64(16))
    tadd = np.uint64(((0x8000 - T) * 0x00010001) & 0xFFFFFFFF)
    g = _u32(w + tadd) & np.uint64(0x80008000)
    np.testing.assert_array_equal((g & np.uint64(0x8000)) != 0, lo >= T)
    np.testing.assert_array_equal((g & np.uint64(0x80000000)) != 0, hi >= T)


def _vmaxu2(a, b):
    lo = np.maximum(a & np.uint64(0xFFFF), b & np.uint64(0xFFFF))
    hi = np.maximum(a >> np.uint64(16), b >> np.uint64(16))
    return lo | (hi << np.uint64(16))


def _perm5432(x, y):
    """__byte_perm(x, y, 0x5432): low half = high half of x, high half = low half of y."""
    return (x >> np.uint64(16)) | ((y & np.uint64(0xFFFF)) << np.uint64(16))


def _pack(c8):
    """8 counts (theta fastest) -> 4 words, word j = (count 2j, count 2j + 1)."""
    c8 = np.asarray(c8, dtype=np.uint64)
    return [c8[2 * j] | (c8[2 * j + 1] << np.uint64(16)) for j in range(4)]


def _chunk_peak_mask(a8, b8, c8, am, bm, cm, ap, bp, cp, T):
    """The kernel's pass-2 arithmetic for one chunk: rows r-1 / r / r+1 (a / b / c), *m = theta row before the chunk,
    *p = theta row after it.  Returns the 8-bit peak mask."""
    A, B, C = _pack(a8), _pack(b8), _pack(c8)
    em = np.uint64(max(am, bm, cm))
    ep = np.uint64(max(ap, bp, cp))
    V = [_vmaxu2(_vmaxu2(A[j], B[j]), C[j]) for j in range(4)]
    Vm = [_perm5432(_u32(em << np.uint64(16)), V[0]), _perm5432(V[0], V[1]), _perm5432(V[1], V[2]), _perm5432(V[2], V[3]),
          _perm5432(V[3], ep)]
    mask = 0
    for j in range(4):
        bh = B[j] | np.uint64(0x80008000)
        sm = _vmaxu2(Vm[j], A[j])
        nm = _vmaxu2(Vm[j + 1], C[j])
        g = _u32(bh - sm - np.uint64(0x00010001)) & _u32(bh - nm) & np.uint64(0x80008000)
        bits = int(((g >> np.uint64(15)) | (g >> np.uint64(30))) & np.uint64(3))
        mask |= bits << (2 * j)
    on = sum(1 << q for q in range(8) if b8[q] >= T)
    return mask & on


@pytest.mark.parametrize("seed,hi", [(0, 4), (1, 40), (2, 1000), (3, 32767)])
def test_packed_local_maximum_test_equals_oracle_peaks(seed, hi):
    """Random small accumulators with many ties; every 8-theta chunk (all positions, borders included) against O4."""
    rng = np.random.default_rng(seed)
    n_theta, n_rho, T = 24, 9, 2
    p = std_params(n_theta, n_rho, T=T)
    for _ in range(12):
        acc = rng.integers(0, hi + 1, (n_theta, n_rho)).astype(np.int64)
        want = set(D.peaks(acc, p))

        def at(t, r):
            return int(acc[t, r]) if 0 <= t < n_theta and 0 <= r < n_rho else 0

        got = set()
        for r in range(n_rho):
            for t0 in range(0, n_theta, 8):
                m = _chunk_peak_mask([at(t0 + q, r - 1) for q in range(8)], [at(t0 + q, r) for q in range(8)],
                                     [at(t0 + q, r + 1) for q in range(8)],
                                     at(t0 - 1, r - 1), at(t0 - 1, r), at(t0 - 1, r + 1),
                                     at(t0 + 8, r - 1), at(t0 + 8, r), at(t0 + 8, r + 1), T)
                got |= {(t0 + q, r) for q in range(8) if (m >> q) & 1}
        assert got == want


def _join_edges(mask, chunk=8):
    """The fast kernel's S3 join rules (hough_fast.cuh, step (c)) on a whole on mask [n_theta][n_rho]: prelinks inside a
    chunk of `chunk` consecutive theta rows, then per on bin at most two explicit joins with neighbours of smaller
    linear index; joins that other joins imply are skipped.  Returns the list of joined pairs."""
    n_theta, n_rho = mask.shape

    def on(t, r):
        return 0 <= t < n_theta and 0 <= r < n_rho and bool(mask[t, r])

    edges = []
    for t in range(n_theta):
        for r in range(n_rho):
            if not mask[t, r]:
                continue
            me = (t, r)
            hoff = on(t - 1, r) and (t % chunk) != 0  # the bin above is on and in the same chunk: prelinked to its run
            if hoff:
                edges.append((me, (t - 1, r)))        # (through the run's head; same component)
            n0, n1, n2, n3 = on(t, r - 1), on(t - 1, r), on(t - 1, r - 1), on(t - 1, r + 1)
            if n1:
                if not hoff:
                    edges.append((me, (t - 1, r)))
                if n0 and not n2:
                    edges.append((me, (t, r - 1)))
            else:
                if n0:
                    edges.append((me, (t, r - 1)))
                elif n2:
                    edges.append((me, (t - 1, r - 1)))
                if n3:
                    edges.append((me, (t - 1, r + 1)))
    return edges


@pytest.mark.parametrize("seed,density", [(0, 0.2), (1, 0.35), (2, 0.5), (3, 0.65), (4, 0.9)])
def test_join_rules_give_the_8_connected_components(seed, density):
    """The pruned joins connect exactly the 8-connected components (scipy.ndimage.label with the 3 x 3 structure), on
    random masks of every density, with chunk seams every 8 theta rows."""
    ndimage = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(seed)
    for _ in range(6):
        mask = rng.random((27, 19)) < density
        parent = {}

        def find(x):
            while parent.setdefault(x, x) != x:
                parent[x] = parent[parent[x]]
                x = parent[x]
            return x

        n_explicit = {}
        for a, b in _join_edges(mask):
            assert mask[a] and mask[b]
            assert max(abs(a[0] - b[0]), abs(a[1] - b[1])) == 1  # only 8-neighbours are ever joined
            n_explicit[a] = n_explicit.get(a, 0) + 1
            ra, rb = find(a), find(b)
            if ra != rb:
                parent[max(ra, rb)] = min(ra, rb)
        assert all(v <= 3 for v in n_explicit.values())  # one prelink + at most two explicit partners
        lab, n = ndimage.label(mask, structure=np.ones((3, 3), dtype=int))
        roots = {}
        for t, r in zip(*np.nonzero(mask)):
            roots.setdefault(find((int(t), int(r))), set()).add(int(lab[t, r]))
        assert len(roots) == n and all(len(s) == 1 for s in roots.values())


def _grid_cases():
    out = [std_params(nt, nr) for nt, nr in [(180, 256), (256, 256), (256, 512), (512, 512), (128, 128), (1024, 1024)]]
    out.append(D.Params(n_theta=180, n_rho=1000, rho_min=-500.0, rho_max=500.0, coord_max=256.0, vote_threshold=24,
                        assign_window=1.0, max_candidates=128))  # the paper's CPU grid
    return out


@pytest.mark.parametrize("p", _grid_cases(), ids=lambda p: f"{p.n_theta}x{p.n_rho}")
def test_safe_radius_and_reachable_rows_bounds(p):
    """Two Cauchy-Schwarz bounds the kernels rely on (hough_lib.cu: r2safe, Mq1; hough_fast.cuh: r_lo, r_hi), checked
    against the exact integer a(h, t) of the definition:
      * u_q^2 + v_q^2 <= r2safe  =>  0 <= a < n_rho 2^F for EVERY theta (such hits vote without a range test);
      * every vote of an event falls into rho rows [(O_q - B) >> F, (O_q + B) >> F], B = (ceil(M) + 1)(ceil(sqrt(r2max)) + 1)."""
    import math
    k = D.constants(p)
    C = np.asarray(k.Cq, dtype=np.int64)
    S = np.asarray(k.Sq, dtype=np.int64)
    top = p.n_rho * (1 << k.F)
    m = min(float(k.Oq), float(top) - 1.0 - float(k.Oq))
    assert m > 0
    R = m / (k.M + 1.0)
    r2safe = int(math.floor(R * R * (1.0 - 1e-9)) - 1.0)
    lim = int(p.coord_max * (1 << k.H))
    rng = np.random.default_rng(11)
    # hits on and just inside the safe circle, at many angles (the extreme a is reached near theta = the hit's own angle)
    ang = np.concatenate([rng.random(3000) * 2 * np.pi, np.linspace(0, 2 * np.pi, 721)])
    rad = math.sqrt(r2safe)
    uq = np.clip(np.trunc(rad * np.cos(ang)).astype(np.int64), -lim, lim)
    vq = np.clip(np.trunc(rad * np.sin(ang)).astype(np.int64), -lim, lim)
    keep = uq * uq + vq * vq <= r2safe
    uq, vq = uq[keep], vq[keep]
    assert uq.size > 1000
    a = uq[:, None] * C[None, :] + vq[:, None] * S[None, :] + k.Oq
    assert a.min() >= 0 and a.max() < top
    # reachable rows of a random event (any valid hits)
    Mq1 = int(math.ceil(k.M)) + 1
    for n in (1, 7, 300):
        eu = rng.integers(-lim, lim + 1, n)
        ev = rng.integers(-lim, lim + 1, n)
        r2max = int((eu * eu + ev * ev).max())
        B = Mq1 * (int(math.ceil(math.sqrt(float(r2max)))) + 1)
        r_lo = max((k.Oq - B) >> k.F, 0)
        r_hi = min((k.Oq + B) >> k.F, p.n_rho - 1)
        rows = (eu[:, None] * C[None, :] + ev[:, None] * S[None, :] + k.Oq) >> k.F
        inr = (rows >= 0) & (rows < p.n_rho)
        assert rows[inr].min() >= r_lo and rows[inr].max() <= r_hi
