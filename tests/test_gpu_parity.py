"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bar (BASELINE.json north_star): relative L2 <= 1e-10, max pointwise relative
<= 1e-9, fp64.  Oracle = oracle/polar_oracle.c (O1 ring-pair direct summation, pinned in
tests/test_oracle_pins.py); inputs = paper_2409_02294_b200.workloads on the library's pg_grid
tables (which are themselves compared with the oracle's tables first)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_2409_02294_b200 import binding as pg
from paper_2409_02294_b200.workloads import CONFIGS, make_batch, make_sigma, random_sigma

pytestmark = pytest.mark.gpu

REL_L2 = 1e-10      # north_star
MAX_REL = 1e-9      # north_star


def errs(got, ref):
    got, ref = np.asarray(got), np.asarray(ref)
    l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got / ref - 1.0).max()
    return l2, mx


def assert_parity(got, ref, what=""):
    l2, mx = errs(got, ref)
    assert l2 <= REL_L2 and mx <= MAX_REL, f"{what}: rel-L2 {l2:.3e} (<= {REL_L2}), max rel {mx:.3e} (<= {MAX_REL})"
    return l2, mx


class Dev:
    """Solver + device buffers held through torch (device memory and stream only)."""

    def __init__(self, n_r, n_phi, r_in, r_out, eps, max_batch=1):
        self.stream = torch.cuda.current_stream()
        self.s = pg.Solver(n_r, n_phi, r_in, r_out, eps, max_batch=max_batch, device=0,
                           cuda_stream=self.stream.cuda_stream)
        self.shape = (n_r, n_phi)

    def solve(self, sigma, direct=False):
        s = np.ascontiguousarray(sigma, dtype=np.float64)
        batch = 1 if s.ndim == 2 else s.shape[0]
        d_s = torch.from_numpy(s).cuda()
        d_p = torch.empty_like(d_s)
        pg.pg_set_density(self.s.h, d_s, batch, pg.PG_MEM_DEVICE)
        (pg.pg_potential_direct if direct else pg.pg_potential)(self.s.h, d_p, batch, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(self.s.h)
        return d_p.cpu().numpy()

    def direct_rings(self, sigma, ring0, n):
        d_s = torch.from_numpy(np.ascontiguousarray(sigma)).cuda()
        d_p = torch.empty((n, self.shape[1]), dtype=torch.float64, device="cuda")
        pg.pg_set_density(self.s.h, d_s, 1, pg.PG_MEM_DEVICE)
        pg.pg_potential_direct_rings(self.s.h, d_p, ring0, n, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(self.s.h)
        return d_p.cpu().numpy()

    def close(self):
        self.s.close()


def cfg_solver(cfg):
    c = CONFIGS[cfg]
    return c, Dev(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, max_batch=c.batch)


# ---------------------------------------------------------------- grid tables (P11 on the GPU side)
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_pg_grid_equals_oracle_grid(cfg):
    c, d = cfg_solver(cfg)
    try:
        r, phi, area = d.s.grid()
        ro, po, ao, _ = oracle.grid(c.n_r, c.n_phi, c.r_in, c.r_out)
        np.testing.assert_allclose(r, ro, rtol=4e-15)
        np.testing.assert_allclose(phi, po, rtol=4e-15)
        np.testing.assert_allclose(area, ao, rtol=2e-13)
    finally:
        d.close()


# ---------------------------------------------------------------- configs 1-2: every cell
@pytest.mark.parametrize("cfg", [1, 2])
def test_fft_path_full_grid_vs_oracle(cfg):
    c, d = cfg_solver(cfg)
    try:
        r, phi, _ = d.s.grid()
        sigma = make_sigma(cfg, r, phi)
        ref = oracle.potential_o1(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma)
        got = d.solve(sigma)
        assert_parity(got, ref, f"config {cfg} FFT path")
        got_d = d.solve(sigma, direct=True)
        assert_parity(got_d, ref, f"config {cfg} direct kernel (a5)")
        assert_parity(got, got_d, f"config {cfg} FFT vs direct on the GPU")
    finally:
        d.close()


# ---------------------------------------------------------------- configs 3-5: sampled target rings at full size
def sample_rings(n_r, n, seed):
    rng = np.random.default_rng(seed)
    fixed = [0, 1, n_r // 2, n_r - 2, n_r - 1]
    extra = rng.choice(np.arange(2, n_r - 2), size=max(0, n - len(fixed)), replace=False)
    return np.unique(np.concatenate([fixed, extra])).astype(np.int32)


@pytest.mark.parametrize("cfg,n_rings", [(3, 48), (5, 10)])
def test_fft_path_sampled_rings_vs_oracle_full_size(cfg, n_rings):
    c, d = cfg_solver(cfg)
    try:
        r, phi, _ = d.s.grid()
        sigma = make_sigma(cfg, r, phi)
        rings = sample_rings(c.n_r, n_rings, cfg)
        ref = oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma, rings)
        got = d.solve(sigma)
        assert np.isfinite(got).all() and (got < 0).all()
        assert_parity(got[rings], ref, f"config {cfg} FFT path, {len(rings)} rings")
        # a5 cross-check on a few of the same rings (direct kernel is O(N^2))
        for i in (0, int(rings[len(rings) // 2]), c.n_r - 1):
            k = int(np.where(rings == i)[0][0])
            gd = d.direct_rings(sigma, i, 1)
            assert_parity(gd[0], ref[k], f"config {cfg} direct kernel ring {i}")
    finally:
        d.close()


def test_config4_batch_of_8_vs_oracle():
    c, d = cfg_solver(4)
    try:
        r, phi, _ = d.s.grid()
        sig = make_batch(4, r, phi)
        assert sig.shape == (8, 1024, 1024)
        got = d.solve(sig)
        for b in range(c.batch):
            rings = sample_rings(c.n_r, 6, 40 + b)
            ref = oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sig[b], rings)
            assert_parity(got[b][rings], ref, f"config 4 field {b}")
        # the batched launch equals eight single solves bit for bit (same kernels, same order)
        one = d.solve(sig[3])
        assert np.array_equal(one, got[3])
    finally:
        d.close()


# ---------------------------------------------------------------- whole grids at the bench sizes
@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_fft_path_vs_direct_kernel_whole_grid(cfg):
    """FFT path (a2-a4) against the direct kernel (a5, from coordinates) on EVERY cell of configs 3, 4 (all eight
    fields) and 5.  a5 itself is tied to the oracle below and in the sampled-ring tests."""
    c, d = cfg_solver(cfg)
    try:
        r, phi, _ = d.s.grid()
        sig = make_batch(cfg, r, phi) if c.batch > 1 else make_sigma(cfg, r, phi)
        got = d.solve(sig)
        ref = d.solve(sig, direct=True)
        if c.batch == 1:
            assert_parity(got, ref, f"config {cfg} FFT vs direct, whole grid")
        else:
            for b in range(c.batch):
                assert_parity(got[b], ref[b], f"config {cfg} field {b} FFT vs direct, whole grid")
    finally:
        d.close()


def sample_targets(n_r, n_phi, n, seed):
    rng = np.random.default_rng(seed)
    rings = np.concatenate([[0, 0, n_r - 1, n_r - 1, n_r // 2], rng.integers(0, n_r, n - 5)])
    cols = rng.integers(0, n_phi, n)
    return (rings.astype(np.int64) * n_phi + cols).astype(np.int64)


def test_direct_kernel_vs_definition_oracle_o0():
    """a5 against O0 -- the four-loop definition from coordinates, NOT the ring-pair oracle O1 whose algorithm
    direct_tiled_kernel mirrors: every cell of config 1, 320 sampled targets of config 5."""
    c, d = cfg_solver(1)
    try:
        r, phi, _ = d.s.grid()
        sigma = make_sigma(1, r, phi)
        ref = oracle.potential_o0(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma)
        assert_parity(d.solve(sigma, direct=True), ref, "config 1 direct kernel vs O0")
    finally:
        d.close()
    c, d = cfg_solver(5)
    try:
        r, phi, _ = d.s.grid()
        sigma = make_sigma(5, r, phi)
        tg = sample_targets(c.n_r, c.n_phi, 320, 55)
        ref = oracle.potential_o0_targets(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma, tg)
        rings = np.unique(tg // c.n_phi)
        got = {int(i): d.direct_rings(sigma, int(i), 1)[0] for i in rings}
        got_t = np.array([got[int(t // c.n_phi)][int(t % c.n_phi)] for t in tg])
        assert_parity(got_t, ref, "config 5 direct kernel vs O0 on sampled targets")
        fft = d.solve(sigma).reshape(-1)[tg]
        assert_parity(fft, ref, "config 5 FFT path vs O0 on sampled targets")
    finally:
        d.close()


def _cached_full_o1(cfg, b, c, sigma):
    """Full-grid O1 of one field, computed once per box and kept in an untracked cache (minutes of CPU)."""
    import hashlib, os, tempfile
    key = hashlib.sha1(sigma.tobytes()).hexdigest()[:16]
    d = os.path.join(tempfile.gettempdir(), "polargrav_oracle_cache")
    os.makedirs(d, exist_ok=True)
    path = os.path.join(d, f"o1_cfg{cfg}_f{b}_{key}.npy")
    if os.path.exists(path):
        return np.load(path)
    ref = oracle.potential_o1(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma)
    np.save(path, ref)
    return ref


@pytest.mark.slow
@pytest.mark.parametrize("cfg", [4, 5])
def test_fft_path_vs_full_grid_oracle_at_bench_sizes(cfg):
    """the parity reference for configs 4-5 is the full-grid O1 result.  Config 5 field 0 (about
    150 s on 16 host threads) and two fields of config 4 (about 10 s each), element by element."""
    c, d = cfg_solver(cfg)
    try:
        r, phi, _ = d.s.grid()
        if cfg == 5:
            sigma = make_sigma(5, r, phi)
            assert_parity(d.solve(sigma), _cached_full_o1(5, 0, c, sigma), "config 5 whole grid vs O1")
        else:
            sig = make_batch(4, r, phi)
            got = d.solve(sig)
            for b in (0, 7):
                assert_parity(got[b], _cached_full_o1(4, b, c, sig[b]), f"config 4 field {b} whole grid vs O1")
    finally:
        d.close()


# ---------------------------------------------------------------- P4 on the GPU: single cell, no wrap-around
@pytest.mark.parametrize("n", [64, 256, 2048])
def test_single_cell_response_no_radial_wraparound(n):
    r_out = {64: 100.0, 256: 500.0, 2048: 2000.0}[n]
    eps = 0.01
    d = Dev(n, n, 1.0, r_out, eps)
    try:
        r, phi, area = d.s.grid()
        h = np.sqrt(area)
        for i0 in (0, n - 1, n // 2):
            j0 = 5
            s = np.zeros((n, n)); s[i0, j0] = 1.0
            d2 = (r[:, None] - r[i0]) ** 2 + 4 * r[:, None] * r[i0] * np.sin(0.5 * (phi[None, :] - phi[j0])) ** 2 \
                + eps ** 2 * h[:, None] * h[i0]
            expect = -area[i0] / np.sqrt(d2)
            got = d.solve(s)
            # rounding of the FFT path is uniform in the reduced potential sqrt(r) Phi
            red = np.abs(got - expect) * np.sqrt(r)[:, None] / np.abs(expect * np.sqrt(r)[:, None]).max()
            assert red.max() <= 1e-13, (n, i0, red.max())
            assert np.abs(got / expect - 1.0).max() <= MAX_REL, (n, i0)
            assert abs(got[i0, j0] / (-h[i0] / eps) - 1.0) <= 1e-12
    finally:
        d.close()


# ---------------------------------------------------------------- invariants at the bench size (hold at any size)
def test_invariants_at_2048():
    c, d = cfg_solver(5)
    try:
        r, phi, area = d.s.grid()
        s1 = make_sigma(5, r, phi)
        p1 = d.solve(s1)
        # P3: roll in phi
        p_roll = d.solve(np.roll(s1, 37, axis=1))
        assert errs(p_roll, np.roll(p1, 37, axis=1))[1] <= 1e-11
        # P2: linearity with a negative weight
        s2 = random_sigma(c.n_r, c.n_phi, 99, signed=True)
        p2 = d.solve(s2)
        p12 = d.solve(0.5 * s1 - 2.0 * s2)
        l2 = np.linalg.norm(p12 - (0.5 * p1 - 2.0 * p2)) / np.linalg.norm(p12)
        assert l2 <= 1e-12
        # P1: axisymmetric density -> axisymmetric potential
        pa = d.solve(np.repeat(np.exp(-r / 200.0)[:, None], c.n_phi, axis=1))
        assert ((pa.max(axis=1) - pa.min(axis=1)) / np.abs(pa).max(axis=1)).max() <= 1e-12
        # P6: reciprocity
        a = (s1 * area[:, None] * p2).sum(); b = (s2 * area[:, None] * p1).sum()
        assert abs(a / b - 1.0) <= 1e-10
    finally:
        d.close()


# ---------------------------------------------------------------- rectangular and small grids
@pytest.mark.parametrize("n_r,n_phi", [(32, 32), (32, 128), (128, 32), (64, 512), (512, 64), (128, 256)])
def test_rectangular_grids_full_vs_oracle(n_r, n_phi):
    d = Dev(n_r, n_phi, 0.7, 60.0, 0.02)
    try:
        s = random_sigma(n_r, n_phi, n_r * 7 + n_phi)
        ref = oracle.potential_o1(n_r, n_phi, 0.7, 60.0, 0.02, s)
        assert_parity(d.solve(s), ref, f"{n_r}x{n_phi} FFT")
        assert_parity(d.solve(s, direct=True), ref, f"{n_r}x{n_phi} direct")
    finally:
        d.close()


def test_zero_density_gives_zero_potential():
    d = Dev(64, 64, 1.0, 100.0, 0.01)
    try:
        assert np.all(d.solve(np.zeros((64, 64))) == 0.0)
    finally:
        d.close()


# ---------------------------------------------------------------- the launch configuration bench.py times
@pytest.mark.parametrize("stable", [0, 1])
@pytest.mark.parametrize("cfg", [3, 5])
def test_back_to_back_solves_equal_isolated_solves(cfg, stable):
    """bench.py enqueues solves back to back on one stream, rotating over distinct (Sigma, Phi) buffers,
    with the kernels chained by programmatic dependent launch (rows_fwd of solve n+1 is scheduled
    while rows_inv of solve n drains, and both use the one W workspace).  Every result of the chain
    must equal, bit for bit, the result of the same solve run alone, and sampled rings must meet the
    oracle at north_star's tolerance."""
    c, d = cfg_solver(cfg)
    try:
        r, phi, _ = d.s.grid()
        base = make_sigma(cfg, r, phi)
        fields = [np.ascontiguousarray(np.roll(base, 37 * k, axis=1) * (1.0 + 0.1 * k)) for k in range(6)]
        alone = [d.solve(f) for f in fields]
        pg.pg_set_option(d.s.h, pg.PG_OPT_DENSITY_STABLE, stable)      # bench.py sets it
        d_s = [torch.from_numpy(f).cuda() for f in fields]
        d_p = [torch.empty_like(t) for t in d_s]
        torch.cuda.synchronize()
        for rep in range(3):                      # 18 solves enqueued without any synchronisation
            for k in range(6):
                pg.pg_set_density(d.s.h, d_s[k], 1, pg.PG_MEM_DEVICE)
                pg.pg_potential(d.s.h, d_p[k], 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(d.s.h)
        for k in range(6):
            assert np.array_equal(d_p[k].cpu().numpy(), alone[k]), f"chained solve {k} differs from the isolated one"
        rings = np.array([0, 1, c.n_r // 2, c.n_r - 1], dtype=np.int32)
        ref = oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, fields[3], rings)
        assert_parity(alone[3][rings], ref, f"config {cfg} chained, sampled rings")
    finally:
        d.close()


def test_partial_batch_uses_the_first_fields_only():
    """A solver created for max_batch = 4 solves batches of 1..4; field b of any batch equals the single solve."""
    d = Dev(128, 256, 1.0, 50.0, 0.01, max_batch=4)
    try:
        fields = np.stack([random_sigma(128, 256, seed=90 + b) for b in range(4)])
        single = [d.solve(fields[b]) for b in range(4)]
        for nb in (1, 2, 3, 4):
            got = d.solve(fields[:nb])
            got = got.reshape(nb, 128, 256)
            for b in range(nb):
                assert np.array_equal(got[b], single[b]), f"batch of {nb}, field {b}"
    finally:
        d.close()


@pytest.mark.parametrize("n_r,n_phi,batch", [(64, 64, 1), (256, 128, 2), (32, 512, 1), (512, 256, 3), (1024, 64, 1),
                                             (64, 2048, 1), (2048, 32, 1), (1024, 1024, 2), (2048, 2048, 1)])
def test_repeated_solves_are_bitwise_reproducible(n_r, n_phi, batch):
    """compute-sanitizer is closed on the GPU pool, so shared-memory hazards (the passes exchange through
    shared memory under named barriers and mbarriers) are hunted this way: 12 repeats of the same solve,
    enqueued back to back, must be identical bit for bit -- a race shows up as run-to-run differences."""
    d = Dev(n_r, n_phi, 1.0, 300.0, 0.01, max_batch=batch)
    try:
        sig = torch.from_numpy(np.stack([random_sigma(n_r, n_phi, seed=700 + b, signed=True) for b in range(batch)])).cuda()
        outs = [torch.empty_like(sig) for _ in range(12)]
        for o in outs:
            pg.pg_set_density(d.s.h, sig, batch, pg.PG_MEM_DEVICE)
            pg.pg_potential(d.s.h, o, batch, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(d.s.h)
        first = outs[0].cpu().numpy()
        assert np.isfinite(first).all()
        for k, o in enumerate(outs[1:], 1):
            assert np.array_equal(o.cpu().numpy(), first), f"repeat {k} differs"
    finally:
        d.close()


def test_potential_fed_back_as_density_with_early_fetch_enabled():
    """PG_OPT_DENSITY_STABLE lets the first kernel of a solve fetch its input while the last kernel of the
    previous solve is still draining.  If the caller (wrongly but plausibly) feeds the previous potential
    straight back as the next density, the library must notice the aliasing and wait: the chain
    Sigma -> Phi1 -> Phi2 -> Phi3 enqueued without synchronisation equals the synchronised one bit for bit."""
    d = Dev(512, 2048, 1.0, 100.0, 0.01)
    try:
        s0 = random_sigma(512, 2048, seed=31)
        p1 = d.solve(s0); p2 = d.solve(p1); p3 = d.solve(p2)
        pg.pg_set_option(d.s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        bufs = [torch.from_numpy(s0).cuda()] + [torch.empty(512, 2048, dtype=torch.float64, device="cuda") for _ in range(3)]
        torch.cuda.synchronize()
        for rep in range(4):
            for k in range(3):
                pg.pg_set_density(d.s.h, bufs[k], 1, pg.PG_MEM_DEVICE)
                pg.pg_potential(d.s.h, bufs[k + 1], 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(d.s.h)
        for got, ref, name in zip(bufs[1:], (p1, p2, p3), ("Phi1", "Phi2", "Phi3")):
            assert np.array_equal(got.cpu().numpy(), ref), name
    finally:
        d.close()


def test_resident_and_staged_solves_interleaved_with_the_option_on():
    """With PG_OPT_DENSITY_STABLE the solver alternates between two W buffers and lets the forward row kernel
    run ahead of the previous solve's last kernel; host-staged solves always use the first buffer and wait.
    Any interleaving of the two kinds, enqueued without synchronisation, must reproduce the isolated results."""
    d = Dev(1024, 512, 1.0, 300.0, 0.01)
    try:
        fields = [random_sigma(1024, 512, seed=40 + k) for k in range(5)]
        alone = [d.solve(f) for f in fields]
        pg.pg_set_option(d.s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        d_s = [torch.from_numpy(f).cuda() for f in fields]
        d_p = [torch.empty_like(t) for t in d_s]
        pin_in, pin_out = pg.PinnedArray((1024, 512)), pg.PinnedArray((1024, 512))
        pin_in.array[...] = fields[4]
        torch.cuda.synchronize()
        pattern = [0, 1, "host", 2, "host", "host", 3, 0, 1, "host", 2, 3]
        for what in pattern:
            if what == "host":
                pg.pg_set_density(d.s.h, pin_in.ptr, 1, pg.PG_MEM_HOST_PINNED)
                pg.pg_potential(d.s.h, pin_out.ptr, 1, pg.PG_MEM_HOST_PINNED)
            else:
                pg.pg_set_density(d.s.h, d_s[what], 1, pg.PG_MEM_DEVICE)
                pg.pg_potential(d.s.h, d_p[what], 1, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(d.s.h)
        for k in range(4):
            assert np.array_equal(d_p[k].cpu().numpy(), alone[k]), f"resident field {k}"
        assert np.array_equal(pin_out.array, alone[4]), "host-staged field"
        pin_in.free(); pin_out.free()
    finally:
        d.close()


@pytest.mark.parametrize("n_r,batch", [(64, 1), (256, 3)])
def test_wide_rows_with_few_rings_and_a_batch(n_r, batch):
    """n_phi = 2048 takes the 4-row row kernels with in-line staging and, in the inverse row kernel, one TMA tile per item
    (tensor map over [field][mode][ring]): few rings (a handful of items per field) and a batch (the field dimension of
    the map) against the oracle on every cell, and the batch against single solves bit for bit."""
    n_phi, r_in, r_out, eps = 2048, 1.0, 40.0, 0.01
    sig = np.stack([random_sigma(n_r, n_phi, 8100 + b) for b in range(batch)])
    s = pg.Solver(n_r, n_phi, r_in, r_out, eps, max_batch=batch, device=0,
                  cuda_stream=torch.cuda.current_stream().cuda_stream)
    try:
        d_s = torch.from_numpy(sig).cuda()
        d_p = torch.empty_like(d_s)
        pg.pg_set_density(s.h, d_s, batch, pg.PG_MEM_DEVICE)
        pg.pg_potential(s.h, d_p, batch, pg.PG_MEM_DEVICE)
        pg.pg_synchronize(s.h)
        got = d_p.cpu().numpy()
        for b in range(batch):
            ref = oracle.potential_o1(n_r, n_phi, r_in, r_out, eps, sig[b])
            assert_parity(got[b], ref, f"{n_r}x{n_phi} field {b}")
            one = torch.empty_like(d_s[b:b + 1])
            pg.pg_set_density(s.h, d_s[b:b + 1].contiguous(), 1, pg.PG_MEM_DEVICE)
            pg.pg_potential(s.h, one, 1, pg.PG_MEM_DEVICE)
            pg.pg_synchronize(s.h)
            assert np.array_equal(one.cpu().numpy()[0], got[b])
    finally:
        s.close()
