"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element,
on the same seeded inputs.  Tolerances are north_star's: relative L2 <= 1e-4 on receiver data and
images, adjoint dot-product test <= 1e-5 (fp32 path; inner products accumulated in fp64)."""
import numpy as np
import pytest

from paper_1709_02733_b200 import synth

pytestmark = pytest.mark.gpu

TOL_L2 = 1e-4     # north_star: GPU (fp32) vs oracle (fp64), relative L2
TOL_DOT = 1e-5    # north_star: adjoint dot-product test of the fp32 path
# Element-wise bars: a norm over 1e8 cells cannot see one wrong cell, row or brick, so every
# comparison also bounds the largest single difference against the largest reference value, and -- for images --
# the difference on every z plane and on every 32 x 32 x (z plane) tile of the fused kernel's decomposition
# against that plane's / tile's own norm (with a floor at the volume's rms level, where "relative" loses meaning).
TOL_MAX = 1e-4    # max |gpu - ref| <= TOL_MAX * max |ref|
TOL_PLANE = 1e-4  # || (gpu - ref)[z] || <= TOL_PLANE * max(|| ref[z] ||, rms plane norm)
TOL_TILE = 2e-4   # the same on 32 x 32 tiles of every plane (fewer cells average less rounding noise)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def closeness(got, ref):
    """rel-L2, max-abs and (3-D arrays) per-plane / per-tile differences of `got` against `ref`, each divided
    by its bar's denominator: every entry must be <= the matching TOL_*."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    d = got - ref
    out = {"l2": float(np.linalg.norm(d) / max(np.linalg.norm(ref), 1e-300)),
           "max": float(np.abs(d).max() / max(np.abs(ref).max(), 1e-300)) if d.size else 0.0}
    if ref.ndim == 3:
        nz, ny, nx = ref.shape
        pn = np.sqrt((ref * ref).sum(axis=(1, 2)))
        floor = np.sqrt((pn * pn).mean())
        out["plane"] = float((np.sqrt((d * d).sum(axis=(1, 2))) / np.maximum(pn, floor)).max())
        ty, tx = -(-ny // 32), -(-nx // 32)
        pad = lambda v: np.pad(v, ((0, 0), (0, ty * 32 - ny), (0, tx * 32 - nx))).reshape(nz, ty, 32, tx, 32)
        tn = np.sqrt((pad(ref) ** 2).sum(axis=(2, 4)))
        tfloor = np.sqrt((tn * tn).mean())
        out["tile"] = float((np.sqrt((pad(d) ** 2).sum(axis=(2, 4))) / np.maximum(tn, tfloor)).max())
    return out


def assert_close(got, ref, what=""):
    c = closeness(got, ref)
    import os
    if os.environ.get("PACT_TEST_LOG"):       # development aid: the measured margins, one JSON line per comparison
        import json
        with open(os.environ["PACT_TEST_LOG"], "a") as fh:
            fh.write(json.dumps({"test": os.environ.get("PYTEST_CURRENT_TEST", ""), "shape": list(np.shape(ref)), **c}) + "\n")
    assert np.isfinite(np.asarray(got)).all(), what
    assert c["l2"] <= TOL_L2, (what, c)
    assert c["max"] <= TOL_MAX, (what, c)
    if "plane" in c:
        assert c["plane"] <= TOL_PLANE and c["tile"] <= TOL_TILE, (what, c)
    return c


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "the gpu-marked tests need a CUDA device"
    from paper_1709_02733_b200 import build
    build.build()
    return torch


def gpu_ops(torch, prob, variant=0, graph=-1, zchunk=0):
    from paper_1709_02733_b200.binding import Pact
    ctx = Pact.from_problem(prob)
    ctx.set_option("variant", variant)
    ctx.set_option("graph", graph)
    ctx.set_option("zchunk", zchunk)
    return ctx


def run_pair(torch, prob, x, y, variant=0, graph=-1, zchunk=0):
    ctx = gpu_ops(torch, prob, variant, graph, zchunk)
    xd = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).cuda()
    yd = torch.from_numpy(np.ascontiguousarray(y, dtype=np.float32)).cuda()
    Hx = ctx.forward(xd).cpu().numpy()
    Hty = ctx.adjoint(yd).cpu().numpy()
    ctx.close()
    return Hx, Hty


def oracle_pair(prob, x, y):
    from oracle.oracle import Oracle
    o = Oracle.from_problem(prob)
    x32 = np.asarray(x, dtype=np.float32).astype(np.float64)   # both sides see the same fp32 inputs
    y32 = np.asarray(y, dtype=np.float32).astype(np.float64)
    Hx, Hty = o.forward(x32), o.adjoint(y32)
    o.close()
    return Hx, Hty


VARIANTS = [1, 2]    # 1: plain two-kernel path ; 2: fused single-pass path (the default)

# sizes span several 32x8x2 (plain) / 32x32 (fused) tiles plus ragged tails in every axis
RANDOM_CASES = [
    dict(nx=45, ny=37, nz=41, nt=40, npml=5, L=19, seed=1, lossy=True),
    dict(nx=70, ny=34, nz=29, nt=30, npml=4, L=11, seed=2, lossy=True),
    dict(nx=33, ny=66, nz=20, nt=25, npml=0, L=9, seed=3, lossy=False),
    dict(nx=75, ny=70, nz=23, nt=22, npml=6, L=13, seed=21, lossy=True),     # 3 x 3 fused tiles, ragged
    dict(nx=100, ny=90, nz=84, nt=16, npml=36, L=9, seed=25, lossy=True),    # C-PML thicker than a tile: whole tiles inside slabs
    dict(nx=8, ny=8, nz=8, nt=12, npml=0, L=3, seed=4, lossy=True),          # minimum grid
    dict(nx=16, ny=17, nz=18, nt=20, npml=4, L=5, seed=5, lossy=True),       # 2*npml+8 == nx: thickest legal PML
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("case", RANDOM_CASES, ids=lambda c: f"{c['nx']}x{c['ny']}x{c['nz']}_p{c['npml']}")
def test_random_heterogeneous_parity_and_dot(torch_cuda, case, variant):
    """Random heterogeneous solid/fluid medium (40 % fluid cells), off-node receivers, random x, y."""
    prob = synth.random_problem(**case)
    x, y = synth.random_vectors(prob, seed=case["seed"])
    Hx, Hty = run_pair(torch_cuda, prob, x, y, variant)
    Hx_o, Hty_o = oracle_pair(prob, x, y)
    assert_close(Hx, Hx_o)
    assert_close(Hty, Hty_o)
    x32, y32 = x.astype(np.float32).astype(np.float64), y.astype(np.float32).astype(np.float64)
    a, b = np.vdot(Hx.astype(np.float64), y32), np.vdot(x32, Hty.astype(np.float64))
    assert abs(a - b) <= TOL_DOT * max(abs(a), abs(b))


@pytest.mark.parametrize("variant", VARIANTS)
def test_config1_full(torch_cuda, variant):
    """BASELINE config 1 at full size (64^3, 300 samples, 128 receivers): forward, adjoint, dot test."""
    prob = synth.make_config(1)
    Hx_o, _ = oracle_pair(prob, prob.p0, np.zeros((prob.prm.nt, prob.L)))
    rng = np.random.default_rng(11)
    y = Hx_o + 0.05 * np.abs(Hx_o).max() * rng.standard_normal(Hx_o.shape)
    Hx, Hty = run_pair(torch_cuda, prob, prob.p0, y, variant)
    _, Hty_o = oracle_pair(prob, np.zeros(prob.p0.shape), y)
    assert_close(Hx, Hx_o)
    assert_close(Hty, Hty_o)
    y32 = y.astype(np.float32).astype(np.float64)
    a, b = np.vdot(Hx.astype(np.float64), y32), np.vdot(prob.p0.astype(np.float64), Hty.astype(np.float64))
    assert abs(a - b) <= TOL_DOT * max(abs(a), abs(b))


@pytest.mark.slow
def test_config2_full_length(torch_cuda):
    """BASELINE config 2 at its full length (128^3, 1000 samples, 512 receivers, absorbing skull shell): fp32 drift
    over 999 steps stays far inside the 1e-4 bar for both kernel families (measured 2e-6 .. 6e-6)."""
    prob = synth.make_config(2)
    rng = np.random.default_rng(5)
    y = rng.standard_normal((prob.prm.nt, prob.L))
    Hx_o, Hty_o = oracle_pair(prob, prob.p0, y)
    for variant in VARIANTS:
        Hx, Hty = run_pair(torch_cuda, prob, prob.p0, y, variant)
        assert_close(Hx, Hx_o)
        assert_close(Hty, Hty_o)


def test_config3_truncated(torch_cuda):
    """BASELINE config 3 (256^3 porous skull, hemispherical array) on its real volumes, 24 samples, automatic
    variant (fused), random x and y: parity and dot test."""
    prob = synth.make_config(3, nt=24)
    x, y = synth.random_vectors(prob, seed=43)
    Hx, Hty = run_pair(torch_cuda, prob, x, y, variant=0)
    Hx_o, Hty_o = oracle_pair(prob, x, y)
    assert_close(Hx, Hx_o)
    assert_close(Hty, Hty_o)
    x32, y32 = x.astype(np.float32).astype(np.float64), y.astype(np.float32).astype(np.float64)
    a, b = np.vdot(Hx.astype(np.float64), y32), np.vdot(x32, Hty.astype(np.float64))
    assert abs(a - b) <= TOL_DOT * max(abs(a), abs(b))


@pytest.mark.parametrize("variant", VARIANTS)
def test_config2_truncated(torch_cuda, variant):
    """BASELINE config 2 (128^3 skull shell, absorption in the shell) on its real volumes, 160 samples."""
    prob = synth.make_config(2, nt=160)
    rng = np.random.default_rng(12)
    y = rng.standard_normal((prob.prm.nt, prob.L))
    Hx, Hty = run_pair(torch_cuda, prob, prob.p0, y, variant)
    Hx_o, Hty_o = oracle_pair(prob, prob.p0, y)
    assert_close(Hx, Hx_o)
    assert_close(Hty, Hty_o)


@pytest.mark.parametrize("zchunk", [1, 5, 16])
def test_fused_z_chunking(torch_cuda, zchunk):
    """The fused kernel marches z in chunks that recompute 2 planes of u on either side: any chunk
    length gives the same operator (several chunks intersect the z slabs of the C-PML here)."""
    prob = synth.random_problem(nx=40, ny=36, nz=45, nt=24, npml=5, L=9, seed=22, lossy=True)
    x, y = synth.random_vectors(prob, seed=22)
    Hx, Hty = run_pair(torch_cuda, prob, x, y, variant=2, zchunk=zchunk)
    Hx_o, Hty_o = oracle_pair(prob, x, y)
    assert_close(Hx, Hx_o)
    assert_close(Hty, Hty_o)


def test_automatic_variant_and_negative_lambda(torch_cuda):
    """variant 0 picks the fused path on a grid with >= 148 bricks of 32^3 and the plain path below;
    a medium with 3 lambda + 2 mu < 0 (legal: lambda + 2 mu > 0) must not take the scaled adjoint."""
    from dataclasses import replace
    prob = synth.random_problem(nx=192, ny=160, nz=170, nt=8, npml=6, L=11, seed=23, lossy=True)   # 6*5*6 = 180 bricks
    x, y = synth.random_vectors(prob, seed=23)
    ctx = gpu_ops(torch_cuda, prob, variant=0, graph=0)
    ctx.set_option("profile", 1)
    xd = torch_cuda.from_numpy(x.astype(np.float32)).cuda()
    Hx = ctx.forward(xd).cpu().numpy()
    _, km, _ = ctx.timing("forward")
    assert km["fwd_slab"] > 0 and km["fwd_interior"] > 0 and km["fwd_vel"] == 0
    ctx.close()
    Hx_o, _ = oracle_pair(prob, x, np.zeros_like(y))
    assert_close(Hx, Hx_o)
    small = synth.random_problem(nx=40, ny=36, nz=33, nt=12, npml=4, L=5, seed=24, lossy=True)
    mu = small.mu.copy(); mu[mu == 0] = mu.max() * 0.1
    aux = replace(small, mu=mu, lam=(-0.8 * mu).astype(np.float32))   # lambda + 2 mu = 1.2 mu > 0 ; 3 lambda + 2 mu < 0
    x, y = synth.random_vectors(aux, seed=24)
    Hx, Hty = run_pair(torch_cuda, aux, x, y, variant=2)               # asks for fused, gets the plain path
    Hx_o, Hty_o = oracle_pair(aux, x, y)
    assert_close(Hx, Hx_o); assert_close(Hty, Hty_o)


def _sign_arrays(seed, k, shape):
    rng = np.random.default_rng(seed)
    return (rng.integers(0, 2, size=(k,) + tuple(shape), dtype=np.int8) * 2 - 1).astype(np.float64)


@pytest.mark.slow
def test_config3_full_length_against_stored_oracle(torch_cuda):
    """BASELINE config 3 at its FULL length (256^3, 2000 samples, 2048 receivers; 1999 steps of the fused kernel)
    against the fp64 oracle's result stored by tests/golden/make_config3_golden.py (a committed script that calls
    only oracle/: the run takes half an hour of CPU, the GPU suite has 20 minutes).  Compared: the full rows of
    every 32nd receiver, random-sign sums over all receivers per time sample (linear in any receiver's error),
    three full-resolution planes of the image, and random-sign sums + norms of every 32 x 32 tile of every z plane
    of the image -- so neither a receiver nor a brick of the decomposition can hide in a norm."""
    import os
    gpath = os.path.join(os.path.dirname(__file__), "golden", "config3_full_oracle.npz")
    G = np.load(gpath)
    prob = synth.make_config(3)
    nt, L = prob.prm.nt, prob.L
    y = np.random.default_rng(int(G["y_seed"])).standard_normal((nt, L)).astype(np.float32)
    ctx = gpu_ops(torch_cuda, prob, variant=0)
    ctx.set_option("check_finite", 1)
    Hx = ctx.forward(torch_cuda.from_numpy(np.ascontiguousarray(prob.p0, dtype=np.float32)).cuda()).cpu().numpy().astype(np.float64)
    Hty = ctx.adjoint(torch_cuda.from_numpy(y).cuda()).cpu().numpy().astype(np.float64)
    ctx.close()
    K = G["data_sums"].shape[1]
    stride = int(G["rcv_stride"])
    # ---- data
    assert_close(Hx[:, ::stride], G["data_rows"], "data rows")
    s = _sign_arrays(int(G["sign_seed"]), K, (L,))
    sums = Hx @ s.T
    scale = np.maximum(G["data_norms"], float(G["data_l2"]) / np.sqrt(nt))[:, None] * 1.0
    assert (np.abs(sums - G["data_sums"]) <= 4 * TOL_L2 * scale).all()       # |sum of L signed errors| <~ ||error|| (x4 margin)
    assert abs(np.linalg.norm(Hx) - float(G["data_l2"])) <= TOL_L2 * float(G["data_l2"])
    # ---- image
    nz, ny, nx = Hty.shape
    amax = float(G["image_absmax"])
    for name, pl in (("image_plane_z", Hty[nz // 2]), ("image_plane_y", Hty[:, ny // 2]), ("image_plane_x", Hty[:, :, nx // 2])):
        ref = G[name].astype(np.float64)
        assert np.abs(pl - ref).max() <= TOL_MAX * amax + 6e-8 * np.abs(ref).max(), name     # + fp32 storage of the golden
        assert rel_l2(pl, ref) <= TOL_L2, name
    s2 = _sign_arrays(int(G["sign_seed"]), K, (ny, nx))
    blk = Hty.reshape(nz, ny // 32, 32, nx // 32, 32)
    tn = G["image_tile_norms"]
    tfloor = np.sqrt((tn * tn).mean())
    for k in range(K):
        sums = (blk * s2[k].reshape(1, ny // 32, 32, nx // 32, 32)).sum(axis=(2, 4))
        assert (np.abs(sums - G["image_tile_sums"][k]) <= 4 * TOL_TILE * np.maximum(tn, tfloor)).all(), k
    norms = np.sqrt((blk * blk).sum(axis=(2, 4)))
    assert (np.abs(norms - tn) <= TOL_TILE * np.maximum(tn, tfloor)).all()
    assert abs(np.linalg.norm(Hty) - float(G["image_l2"])) <= TOL_L2 * float(G["image_l2"])


@pytest.mark.slow
@pytest.mark.parametrize("k", [4, 5])
def test_config4_config5_real_volumes_50_steps(torch_cuda, k):
    """BASELINE configs 4 (512^3, 16-cell C-PML, 4096 receivers) and 5 (384^3, 2048 receivers) at full size on
    their real volumes (porous skull), in the launch configuration bench.py times (automatic variant = fused, no
    graph), 51 samples = 50 steps (">= 50 steps"; the oracle takes minutes).  Random x over the whole
    grid and random y, so the C-PML slabs and every receiver carry signal.  Element-wise, per-plane and per-tile
    bars besides the norm, and the dot test."""
    prob = synth.make_config(k, nt=51)
    x, y = synth.random_vectors(prob, seed=40 + k)
    ctx = gpu_ops(torch_cuda, prob, variant=0)
    ctx.set_option("profile", 1)
    ctx.set_option("check_finite", 1)
    xd = torch_cuda.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).cuda()
    yd = torch_cuda.from_numpy(np.ascontiguousarray(y, dtype=np.float32)).cuda()
    Hx = ctx.forward(xd).cpu().numpy()
    Hty = ctx.adjoint(yd).cpu().numpy()
    _, km, _ = ctx.timing("adjoint")
    assert km["adj_slab"] > 0 and km["adj_interior"] > 0      # the fused kernel is what ran, on both kinds of brick
    ctx.close()
    del xd, yd
    Hx_o, Hty_o = oracle_pair(prob, x, y)
    assert_close(Hx, Hx_o)
    assert_close(Hty, Hty_o)
    x32, y32 = x.astype(np.float32).astype(np.float64), y.astype(np.float32).astype(np.float64)
    a, b = np.vdot(Hx.astype(np.float64), y32), np.vdot(x32, Hty.astype(np.float64))
    assert abs(a - b) <= TOL_DOT * max(abs(a), abs(b))


def test_fused_is_bitwise_repeatable(torch_cuda):
    """The fused kernel synchronises with one block barrier per plane plus mbarriers, re-uses shared-memory slots
    as soon as their last reader has passed a barrier, and runs interior and slab bricks on two streams: a missed
    hazard would show up as run-to-run differences.  Five runs of H and H^T on a 3 x 3 tile grid with several z
    chunks (x, y and z slabs, corner tiles) must agree bit for bit.  (compute-sanitizer is closed on this pool.)"""
    torch = torch_cuda
    prob = synth.random_problem(nx=90, ny=75, nz=50, nt=14, npml=7, L=17, seed=31, lossy=True)
    x, y = synth.random_vectors(prob, seed=31)
    ctx = gpu_ops(torch, prob, variant=2, graph=0, zchunk=9)
    xd, yd = torch.from_numpy(x.astype(np.float32)).cuda(), torch.from_numpy(y.astype(np.float32)).cuda()
    d0, i0 = ctx.forward(xd).clone(), ctx.adjoint(yd).clone()
    for _ in range(4):
        assert torch.equal(ctx.forward(xd), d0)
        assert torch.equal(ctx.adjoint(yd), i0)
    ctx.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_graph_and_direct_launch_agree_bitwise(torch_cuda, variant):
    """The time loop replayed from a captured CUDA graph (for the fused path the capture includes the fork to the
    second stream and the join) gives the same bits as direct launches."""
    prob = synth.random_problem(nx=72, ny=70, nz=33, nt=30, npml=4, L=7, seed=6)     # 3 x 3 tiles: interior + slab lists
    x, y = synth.random_vectors(prob, seed=6)
    a = run_pair(torch_cuda, prob, x, y, variant=variant, graph=1)
    b = run_pair(torch_cuda, prob, x, y, variant=variant, graph=0)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_fused_without_receivers(torch_cuda):
    """L = 0 on the fused path: empty data, zero image."""
    torch = torch_cuda
    from dataclasses import replace
    prob = synth.random_problem(nx=40, ny=36, nz=34, nt=9, npml=3, L=4, seed=12, lossy=True)
    ctx = gpu_ops(torch, replace(prob, rcv=np.zeros((0, 3))), variant=2)
    x, _ = synth.random_vectors(prob, seed=12)
    assert ctx.forward(torch.from_numpy(x.astype(np.float32)).cuda()).shape == (prob.prm.nt, 0)
    img = ctx.adjoint(torch.empty((prob.prm.nt, 0), dtype=torch.float32, device="cuda"))
    assert float(img.abs().max()) == 0.0
    ctx.close()


def test_calls_are_repeatable_and_independent(torch_cuda):
    """Each call resets the state: forward, adjoint, forward again gives bit-identical data."""
    torch = torch_cuda
    prob = synth.random_problem(nx=24, ny=20, nz=28, nt=20, npml=4, L=6, seed=7)
    x, y = synth.random_vectors(prob, seed=7)
    ctx = gpu_ops(torch, prob)
    xd, yd = torch.from_numpy(x.astype(np.float32)).cuda(), torch.from_numpy(y.astype(np.float32)).cuda()
    d1 = ctx.forward(xd).clone()
    i1 = ctx.adjoint(yd).clone()
    d2 = ctx.forward(xd)
    i2 = ctx.adjoint(yd)
    assert torch.equal(d1, d2) and torch.equal(i1, i2)
    ctx.close()


def test_host_buffer_entry_points(torch_cuda):
    torch = torch_cuda
    prob = synth.random_problem(nx=24, ny=20, nz=28, nt=20, npml=4, L=6, seed=8)
    x, y = synth.random_vectors(prob, seed=8)
    ctx = gpu_ops(torch, prob)
    xh = torch.from_numpy(x.astype(np.float32)).pin_memory()
    yh = torch.from_numpy(y.astype(np.float32)).pin_memory()
    dh = torch.empty((prob.prm.nt, prob.L), dtype=torch.float32).pin_memory()
    ih = torch.empty(prob.p0.shape, dtype=torch.float32).pin_memory()
    ctx.forward_host(xh, dh)
    ctx.adjoint_host(yh, ih)
    assert torch.equal(dh, ctx.forward(xh.cuda()).cpu())
    assert torch.equal(ih, ctx.adjoint(yh.cuda()).cpu())
    ctx.close()


def test_error_codes(torch_cuda):
    torch = torch_cuda
    from dataclasses import replace
    from paper_1709_02733_b200.binding import Pact, PactError
    prob = synth.random_problem(nx=16, ny=16, nz=16, nt=5, npml=2, L=3, seed=9)
    with pytest.raises(PactError) as e:   # dt above the stability limit
        Pact.from_problem(replace(prob, prm=replace(prob.prm, dt=prob.prm.dt * 3.0)))
    assert e.value.code == -2
    bad = prob.rcv.copy(); bad[0, 0] = -prob.prm.h
    with pytest.raises(PactError) as e:   # receiver outside the grid
        Pact.from_problem(replace(prob, rcv=bad))
    assert e.value.code == -3
    rho = prob.rho.copy(); rho[3, 4, 5] = 0.0
    with pytest.raises(PactError) as e:   # rho <= 0
        Pact.from_problem(replace(prob, rho=rho))
    assert e.value.code == -4
    lam = prob.lam.copy(); lam[0, 0, 0] = np.nan
    with pytest.raises(PactError) as e:
        Pact.from_problem(replace(prob, lam=lam))
    assert e.value.code == -4
    with pytest.raises(PactError) as e:   # PML too thick for the grid
        Pact.from_problem(replace(prob, prm=replace(prob.prm, npml=5)))
    assert e.value.code == -1


def test_no_receivers_and_lossless_null_alpha(torch_cuda):
    """L = 0 is legal (data is empty, image is zero); alpha = NULL means lossless."""
    torch = torch_cuda
    from dataclasses import replace
    from paper_1709_02733_b200.binding import Pact
    prob = synth.random_problem(nx=20, ny=18, nz=16, nt=15, npml=3, L=4, seed=10, lossy=False)
    x, y = synth.random_vectors(prob, seed=10)
    a = Pact.from_problem(prob)
    b = Pact.from_problem(replace(prob, alpha=None))
    xd = torch.from_numpy(x.astype(np.float32)).cuda()
    assert torch.equal(a.forward(xd), b.forward(xd))
    c = Pact.from_problem(replace(prob, rcv=np.zeros((0, 3))))
    assert c.forward(xd).shape == (prob.prm.nt, 0)
    img = c.adjoint(torch.empty((prob.prm.nt, 0), dtype=torch.float32, device="cuda"))
    assert float(img.abs().max()) == 0.0
    for k in (a, b, c):
        k.close()


def test_single_persistent_launch_equals_split_launches(torch_cuda):
    """A fused time step runs as two launches (C-PML bricks, then C-PML-free bricks: the default, each timed on its
    own) or as one persistent launch over the whole work list (option split_launch = 0): same bricks, same bits."""
    torch = torch_cuda
    prob = synth.random_problem(nx=100, ny=98, nz=60, nt=12, npml=5, L=9, seed=33, lossy=True)   # 4 x 4 tiles: 4 interior
    x, y = synth.random_vectors(prob, seed=33)
    xd, yd = torch.from_numpy(x.astype(np.float32)).cuda(), torch.from_numpy(y.astype(np.float32)).cuda()
    res = []
    for split in (1, 0):
        ctx = gpu_ops(torch, prob, variant=2, graph=0)
        ctx.set_option("split_launch", split)
        ctx.set_option("profile", 1)
        res.append((ctx.forward(xd).clone(), ctx.adjoint(yd).clone()))
        _, km, ln = ctx.timing("adjoint")
        assert (km["adj_fused"] > 0) == (split == 0) and (km["adj_slab"] > 0) == (split == 1)
        ctx.close()
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])


def test_check_finite_reports_a_blow_up(torch_cuda):
    """Option check_finite (failure detection): a NaN in the result comes back as PACT_ENUMERIC
    from both operators and both kernel families; finite results pass."""
    torch = torch_cuda
    from paper_1709_02733_b200.binding import PactError
    prob = synth.random_problem(nx=40, ny=36, nz=34, nt=9, npml=3, L=4, seed=13, lossy=True)
    x, y = synth.random_vectors(prob, seed=13)
    for variant in VARIANTS:
        ctx = gpu_ops(torch, prob, variant=variant)
        ctx.set_option("check_finite", 1)
        xd, yd = torch.from_numpy(x.astype(np.float32)).cuda(), torch.from_numpy(y.astype(np.float32)).cuda()
        ctx.forward(xd); ctx.adjoint(yd)                       # finite: no error
        xd[prob.prm.nz // 2, prob.prm.ny // 2, prob.prm.nx // 2] = float("nan")
        yd[3, 1] = float("inf")
        with pytest.raises(PactError) as e:
            ctx.forward(xd)
        assert e.value.code == -7
        with pytest.raises(PactError) as e:
            ctx.adjoint(yd)
        assert e.value.code == -7
        ctx.set_option("check_finite", 0)
        ctx.forward(xd)                                        # unchecked: no error, asynchronous
        ctx.close()


def test_pml_constants_default_when_zero(torch_cuda):
    """include/pact.h: pml_R = 0 selects 1e-4, pml_cref = 0 selects max c_l of the medium."""
    torch = torch_cuda
    from dataclasses import replace
    prob = synth.random_problem(nx=24, ny=20, nz=28, nt=10, npml=4, L=6, seed=14)
    cmax = float(np.sqrt(((prob.lam.astype(np.float64) + 2 * prob.mu) / prob.rho).max()))
    x, _ = synth.random_vectors(prob, seed=14)
    xd = torch.from_numpy(x.astype(np.float32)).cuda()
    a = gpu_ops(torch, replace(prob, prm=replace(prob.prm, pml_R=0.0, pml_cref=0.0)))
    b = gpu_ops(torch, replace(prob, prm=replace(prob.prm, pml_R=1e-4, pml_cref=cmax)))
    da, db = a.forward(xd), b.forward(xd)
    assert rel_l2(da.cpu().numpy(), db.cpu().numpy()) <= 1e-6      # c_max is found in fp32 on the device
    a.close(); b.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_long_run_at_the_stability_limit(torch_cuda, variant):
    """PACT_ECFL checks the nodal bound only (include/pact.h).  A water / skull-shell medium (density contrast
    1.85, arithmetic staggered densities) run at 0.99 of that bound for 1500 steps with noise that
    excites every mode stays bounded on the GPU as it does in the oracle (tests/test_oracle_pins.py)."""
    torch = torch_cuda
    from dataclasses import replace
    n, h = 40, 0.2e-3
    prm0 = synth.Params(n, n, n, h, 1.0, 1500, 4)
    r = synth.radius_field(prm0, synth.centre(prm0))
    shell = (r > 1.8e-3) & (r < 2.6e-3)
    cp, cs, rho = np.where(shell, 3000.0, 1500.0), np.where(shell, 1500.0, 0.0), np.where(shell, 1850.0, 1000.0)
    prm = replace(prm0, dt=synth.stable_dt(h, 3000.0, 0.99), pml_cref=3000.0)
    p0 = np.random.default_rng(5).standard_normal((n, n, n))
    rcv = synth.centre(prm)[None, :] + 0.3e-3
    pb = synth.custom_problem("stab", prm, cp, cs, rho, 0.0, rcv, p0)
    ctx = gpu_ops(torch, pb, variant=variant)
    ctx.set_option("check_finite", 1)
    d = ctx.forward(torch.from_numpy(pb.p0.astype(np.float32)).cuda()).cpu().numpy()
    ctx.close()
    assert np.abs(d[-200:]).max() <= 10 * np.abs(d[:200]).max()


def test_material_elision_is_bit_exact(torch_cuda):
    """Homogeneous (tile, plane) material boxes are fetched from a palette plane instead of their own plane
    (DESIGN.md "Homogeneous material planes"): config 2 has two homogeneous media (water, brain) around a shell, so
    most planes are elided -- and the operator must not change by a bit against the run that fetches every plane."""
    torch = torch_cuda
    prob = synth.make_config(2, nt=40)
    y = np.random.default_rng(15).standard_normal((prob.prm.nt, prob.L)).astype(np.float32)
    xd, yd = torch.from_numpy(prob.p0.astype(np.float32)).cuda(), torch.from_numpy(y).cuda()
    out = []
    for elide in (1, 0):
        ctx = gpu_ops(torch, prob, variant=2, graph=0)
        ctx.set_option("material_elision", elide)
        if elide:
            assert ctx.info("elided_material_planes") > 0.3
        out.append((ctx.forward(xd).clone(), ctx.adjoint(yd).clone()))
        ctx.close()
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])
    # a random heterogeneous medium has nothing to elide
    rp = synth.random_problem(nx=40, ny=36, nz=34, nt=4, npml=3, L=4, seed=16, lossy=True)
    ctx = gpu_ops(torch, rp, variant=2)
    assert ctx.info("elided_material_planes") == 0.0
    ctx.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_projected_gradient_matches_oracle(torch_cuda, variant):
    """power-iteration step size and three projected-gradient iterations
    p <- max(0, p - s H^T (H p - d)) through pact_power_iteration / pact_pgd against the same recursion on the fp64
    oracle (oracle/pgd.py): step size to 1e-4, every iterate, residual norm and update norm to 1e-4."""
    torch = torch_cuda
    from oracle.oracle import Oracle
    from oracle import pgd as opgd
    prob = synth.random_problem(nx=44, ny=40, nz=36, nt=60, npml=5, L=24, seed=51, lossy=True)
    rng = np.random.default_rng(51)
    p_true = np.maximum(rng.standard_normal(prob.p0.shape), 0.0) * (rng.random(prob.p0.shape) < 0.05)
    v0 = rng.standard_normal(prob.p0.shape).astype(np.float32)
    o = Oracle.from_problem(prob)
    d = o.forward(p_true.astype(np.float32).astype(np.float64))
    d = (d + 0.01 * np.abs(d).max() * rng.standard_normal(d.shape)).astype(np.float32)
    s2_o, _ = opgd.power_iteration(o, v0.astype(np.float64), iters=6)
    its_o, res_o, upd_o = opgd.pgd(o, np.zeros(prob.p0.shape), d.astype(np.float64), 1.0 / s2_o, 3)
    o.close()
    ctx = gpu_ops(torch, prob, variant=variant)
    ctx.set_option("check_finite", 1)
    vd = torch.from_numpy(v0).cuda()
    s2 = ctx.power_iteration(vd, iters=6)
    assert abs(s2 - s2_o) <= 1e-4 * s2_o
    assert abs(float(vd.double().norm()) - 1.0) <= 1e-5
    dd = torch.from_numpy(d).cuda()
    p = torch.zeros(ctx.shape, dtype=torch.float32, device="cuda")
    for k in range(3):             # one iteration per call, so that every iterate can be compared
        res, upd = ctx.pgd(p, dd, 1.0 / s2_o, 1)
        assert_close(p.cpu().numpy(), its_o[k], f"iterate {k + 1}")
        assert abs(res[0] - res_o[k]) <= 1e-4 * res_o[k] and abs(upd[0] - upd_o[k]) <= 1e-4 * upd_o[k]
        assert float(p.min()) >= 0.0
    # the same three iterations in one call give the same bits, and the residual decreases
    p2 = torch.zeros_like(p)
    res3, _ = ctx.pgd(p2, dd, 1.0 / s2_o, 3)
    assert torch.equal(p, p2) and res3[0] > res3[1] > res3[2]
    ctx.close()


ACOUSTIC_CASES = [
    dict(nx=75, ny=70, nz=40, nt=30, npml=6, L=13, seed=61, lossy=True),      # 3 x 3 tiles, ragged, every brick touches a slab
    dict(nx=130, ny=100, nz=64, nt=20, npml=5, L=9, seed=62, lossy=True),     # 5 x 4 tiles with C-PML-free bricks
    dict(nx=40, ny=36, nz=33, nt=16, npml=0, L=5, seed=63, lossy=False),      # no C-PML, lossless
]


@pytest.mark.parametrize("case", ACOUSTIC_CASES, ids=lambda c: f"{c['nx']}x{c['ny']}x{c['nz']}_p{c['npml']}")
def test_fluid_medium_takes_the_acoustic_kernels(torch_cuda, case):
    """SURVEY 8(f)-2 (the paper's H^dagger_{mu=0}): a medium with mu = 0 everywhere runs the
    fluid-only kernel pair of the fused path (one stress field + three velocities).  Parity and dot test against
    the oracle run with mu = 0 (itself pinned against textbook acoustics), and agreement to rounding with the
    elastic kernels on the same medium (option acoustic = 0)."""
    torch = torch_cuda
    prob = synth.random_problem(fluid_fraction=1.0, **case)
    assert not prob.mu.any()
    x, y = synth.random_vectors(prob, seed=case["seed"])
    xd, yd = torch.from_numpy(x.astype(np.float32)).cuda(), torch.from_numpy(y.astype(np.float32)).cuda()
    ctx = gpu_ops(torch, prob, variant=2, graph=0)
    assert ctx.info("fluid") == 1.0 and ctx.info("acoustic_path") == 1.0
    Hx, Hty = ctx.forward(xd).clone(), ctx.adjoint(yd).clone()
    ctx.set_option("acoustic", 0)
    assert ctx.info("acoustic_path") == 0.0
    # the elastic kernels on the same medium: the same numbers up to the last bit of a few roundings (measured: 1-2 ulp)
    for got, ref in ((Hx, ctx.forward(xd)), (Hty, ctx.adjoint(yd))):
        assert float((got - ref).abs().max()) <= 2e-6 * float(ref.abs().max())
    ctx.close()
    Hx_o, Hty_o = oracle_pair(prob, x, y)
    assert_close(Hx.cpu().numpy(), Hx_o)
    assert_close(Hty.cpu().numpy(), Hty_o)
    x32, y32 = x.astype(np.float32).astype(np.float64), y.astype(np.float32).astype(np.float64)
    a, b = np.vdot(Hx.cpu().numpy().astype(np.float64), y32), np.vdot(x32, Hty.cpu().numpy().astype(np.float64))
    assert abs(a - b) <= TOL_DOT * max(abs(a), abs(b))
    # a medium with any solid cell keeps the elastic kernels
    solid = synth.random_problem(nx=40, ny=36, nz=33, nt=4, npml=3, L=4, seed=64)
    c2 = gpu_ops(torch, solid, variant=2)
    assert c2.info("fluid") == 0.0 and c2.info("acoustic_path") == 0.0
    c2.close()
