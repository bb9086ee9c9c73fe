"""GPU parity: the CUDA path (through the C-ABI, via the ctypes binding) against the fp64 oracle,
element by element, on the same seeded inputs.

Bars (BASELINE.json north_star):
  * remap permutation and remapped tensor copy: bit-exact against the oracle's stable sort;
  * Y_d: max |Y_gpu - Y_oracle| / S_d <= 1e-5 with S_d = sum |val| prod |A_m| per entry, and entries
    with S_d == 0 exactly 0.
"""
import numpy as np
import pytest
import torch

import oracle
import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def P():
    import paper_2405_08470_b200 as pkg
    pkg.load_library()          # fails loudly if the CUDA library is missing
    assert torch.cuda.is_available()
    return pkg


def _run_case(P, dims, idx_cpu, vals_cpu, R, seed, order_modes=None, check_perm=True, ones=False):
    N = len(dims)
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(seed)
    if ones:
        fac_np = [np.ones((d, R), dtype=np.float32) for d in dims]
    else:
        fac_np = [rng.uniform(-1, 1, size=(d, R)).astype(np.float32) for d in dims]
    fac = [torch.from_numpy(f).to(dev) for f in fac_np]
    h = P.Mttkrp(dims, idx_cpu.to(dev), vals_cpu.to(dev))
    info = h.info()
    assert info["cur_layout"] == 0 and info["nnz"] == vals_cpu.numel()
    idx_np, vals_np = idx_cpu.numpy(), vals_cpu.numpy()
    perms = {}
    if check_perm and vals_cpu.numel() > 0:
        for d in range(N):
            order = info["key_order"][d]
            assert order[0] == d and sorted(order) == list(range(N))
            perms[d] = oracle.sort_perm(dims, idx_np, order)
            got = h.get_perm(d).cpu().numpy().astype(np.int64)
            np.testing.assert_array_equal(got, perms[d])            # bit-exact (Observation 1: a bijection)
    modes = list(order_modes) if order_modes is not None else list(range(N))
    worst = 0.0
    for d in modes:
        out = torch.full((dims[d], R), float("nan"), dtype=torch.float32, device=dev)   # every entry must be overwritten
        Y = h.mttkrp_mode(d, fac, out=out).cpu().numpy()
        assert h.info()["cur_layout"] == d
        if d in perms:                                                # remapped copy is the sorted COO
            gi, gv = h.export_coo()
            np.testing.assert_array_equal(gi.cpu().numpy(), idx_np[:, perms[d]])
            np.testing.assert_array_equal(gv.cpu().numpy(), vals_np[perms[d]])
        Yo, So = oracle.mttkrp_mode(dims, idx_np, vals_np, fac_np, d, perm=perms.get(d))
        err, zeros_ok = oracle.normalised_error(Y, Yo, So)
        assert zeros_ok, f"mode {d}: entries without contributions must be exactly 0"
        assert err <= TOL, f"mode {d}: normalised error {err:.3e} > {TOL}"
        worst = max(worst, err)
    h.destroy()
    return worst, info


@pytest.mark.parametrize("dims,nnz,dup", [((4, 3, 5), 30, False), ((3, 4, 2, 3), 40, True), ((2, 3, 2, 2, 3), 50, False),
                                          ((5, 4), 12, True), ((7, 1, 3), 15, False), ((2, 2, 2, 2, 2, 2), 40, True),
                                          ((3, 2, 2, 2, 2, 2, 2), 60, True), ((2, 2, 2, 3, 2, 2, 2, 2), 80, True)])
@pytest.mark.parametrize("R", [8, 32])
def test_tiny_tensors(P, dims, nnz, dup, R):
    t = W.tiny_tensor(dims, nnz, seed=len(dims) * 100 + nnz, duplicates=dup)
    _run_case(P, list(dims), t.idx, t.vals, R, seed=1)


def test_hand_worked_golden(P):
    # tests/golden/hand_worked_3mode.txt (PAPER.md:121 by hand); rank 2 is padded to the library's smallest
    # rank with zero columns.  Small integers and halves: exact in fp32.
    from conftest import load_golden
    dims, idx, vals, factors, want = load_golden("hand_worked_3mode.txt")
    dev = torch.device("cuda:0")
    fac = [torch.from_numpy(np.pad(f, ((0, 0), (0, 6)))).to(dev) for f in factors]
    h = P.Mttkrp(dims, torch.from_numpy(idx).to(dev), torch.from_numpy(vals).to(dev))
    for d in [0, 1, 2, 1]:
        Y = h.mttkrp_mode(d, fac).cpu().numpy()
        np.testing.assert_array_equal(Y[:, :2].astype(np.float64), want[d])
        assert np.all(Y[:, 2:] == 0)
    h.destroy()


@pytest.mark.parametrize("R", [8, 16, 32, 64])
def test_config1_full(P, R):
    # BASELINE.json configs[0] at full size (R=16 is the config's rank; the others widen it).
    spec = W.CONFIGS[0]
    t = W.generate_tensor(spec)
    worst, info = _run_case(P, spec.dims, t.idx, t.vals, R, seed=2)
    assert info["num_shards"] > 1


@pytest.mark.parametrize("cfg,nnz,R", [(1, 300_000, 32), (2, 300_000, 32), (3, 250_000, 32), (4, 200_000, 8),
                                       (4, 200_000, 16), (4, 200_000, 32), (4, 200_000, 64)])
def test_scaled_configs(P, cfg, nnz, R):
    # Shape classes of configs 2-5 (Zipf skew, tiny and huge modes) at sizes the oracle does in
    # seconds; nnz is not a multiple of the shard size (ragged tail) and spans many shards.
    spec = W.CONFIGS[cfg].scaled(nnz + 137)
    t = W.generate_tensor(spec)
    worst, info = _run_case(P, spec.dims, t.idx, t.vals, R, seed=3)
    assert info["num_shards"] >= 30
    assert max(info["num_split_rows"]) > 0          # skewed modes do have rows spanning shards


def test_heavy_rows_span_many_shards(P):
    # Degenerate: a mode with 2 rows (the paper's Vast tensor has one) and a mode of size 1.
    dims = [2, 50, 1, 400]
    spec = W.TensorSpec("heavy", dims, 30_000, [0.0, 0.0, 0.0, 0.0], "uniform", (32,), 77)
    t = W.generate_tensor(spec)
    worst, info = _run_case(P, dims, t.idx, t.vals, 32, seed=4)
    assert info["num_split_rows"][0] >= 1 and info["num_split_rows"][2] == 1


def test_all_ones_closed_form(P):
    # All-ones dense tensor and factors: Y_d[i, r] = prod_{m != d} I_m exactly (fp32 below 2^24).
    dims = [12, 9, 11]
    grid = np.stack(np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")).reshape(3, -1).astype(np.int32)
    rng = np.random.default_rng(0)
    grid = grid[:, rng.permutation(grid.shape[1])]
    idx = torch.from_numpy(np.ascontiguousarray(grid))
    vals = torch.ones(idx.shape[1], dtype=torch.float32)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(dims, idx.to(dev), vals.to(dev))
    fac = [torch.ones((d, 16), dtype=torch.float32, device=dev) for d in dims]
    for d in range(3):
        Y = h.mttkrp_mode(d, fac).cpu().numpy()
        want = np.prod([dims[m] for m in range(3) if m != d])
        assert np.all(Y == float(want))
    h.destroy()


def test_any_order_and_repeat(P):
    # Layouts are history-free (reading 5): any call order gives the same result.
    spec = W.CONFIGS[0].scaled(20_011)
    t = W.generate_tensor(spec)
    _run_case(P, spec.dims, t.idx, t.vals, 16, seed=5, order_modes=[2, 2, 0, 1, 0, 2, 1, 1], check_perm=True)


def test_empty_tensor_and_empty_rows(P):
    dev = torch.device("cuda:0")
    dims = [5, 4, 3]
    h = P.Mttkrp(dims, torch.empty((3, 0), dtype=torch.int32, device=dev), torch.empty(0, dtype=torch.float32, device=dev))
    fac = [torch.rand((d, 8), device=dev) for d in dims]
    for d in range(3):
        out = torch.full((dims[d], 8), float("nan"), device=dev)
        h.mttkrp_mode(d, fac, out=out)
        assert torch.all(out == 0)
    assert h.info()["num_empty_rows"] == dims
    h.destroy()
    # one nonzero in a large mode: every other row must be overwritten with zeros (NaN-poisoned out)
    dims = [1000, 3, 2]
    idx = torch.tensor([[777], [1], [0]], dtype=torch.int32, device=dev)
    vals = torch.tensor([2.0], device=dev)
    h = P.Mttkrp(dims, idx, vals)
    fac = [torch.full((d, 32), 0.5, device=dev) for d in dims]
    out = torch.full((1000, 32), float("nan"), device=dev)
    h.mttkrp_mode(0, fac, out=out)
    assert torch.all(out[777] == 0.5) and torch.all(out[:777] == 0) and torch.all(out[778:] == 0)
    h.destroy()


def test_sweep_and_host_entry_points(P):
    spec = W.CONFIGS[0].scaled(50_021)
    t = W.generate_tensor(spec)
    dev = torch.device("cuda:0")
    R = 16
    fac_cpu = W.generate_factors(spec, R)
    fac = [f.to(dev) for f in fac_cpu]
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev), max_rank=R)
    outs = h.mttkrp_sweep(fac)
    fac_pin = [f.pin_memory() for f in fac_cpu]
    outs_host = [torch.empty((d, R), dtype=torch.float32).pin_memory() for d in spec.dims]
    h.mttkrp_sweep_host(fac_pin, outs_host)
    for d in range(3):
        assert torch.equal(outs[d].cpu(), outs_host[d])            # same kernels, same order: bit-identical
        Yo, So = oracle.mttkrp_mode(spec.dims, t.idx.numpy(), t.vals.numpy(), [f.numpy() for f in fac_cpu], d)
        err, zeros_ok = oracle.normalised_error(outs[d].cpu().numpy(), Yo, So)
        assert zeros_ok and err <= TOL
    assert h.info()["remaps_done"] == 5          # 0->1->2 (sweep), 2->0->1->2 (host sweep): 2 + 3
    h.destroy()


def test_side_stream_and_changing_rank(P):
    # The library works on whatever stream the caller passes (the binding passes torch's current stream) and
    # keeps no per-rank state: R may change from call to call.
    spec = W.CONFIGS[0].scaled(30_011)
    t = W.generate_tensor(spec)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
    ref = {}
    for R in (8, 32):
        fac = [f.to(dev) for f in W.generate_factors(spec, R)]
        ref[R] = [y.clone() for y in h.mttkrp_sweep(fac)]
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        for R in (32, 8, 32):
            fac = [f.to(dev) for f in W.generate_factors(spec, R)]
            outs = h.mttkrp_sweep(fac)
            side.synchronize()
            for d in range(3):
                assert torch.equal(outs[d], ref[R][d])          # same kernels, same order: bit-identical
    h.destroy()


def test_errors_are_reported(P):
    dev = torch.device("cuda:0")
    dims = [5, 4, 3]
    idx = torch.tensor([[0, 5], [1, 1], [2, 2]], dtype=torch.int32, device=dev)      # 5 is out of range in mode 0
    vals = torch.ones(2, device=dev)
    with pytest.raises(P.MttkrpError) as e:
        P.Mttkrp(dims, idx, vals)
    assert e.value.status == 2          # MTTKRP_EINDEX
    idx[0, 1] = 4
    h = P.Mttkrp(dims, idx, vals)
    fac = [torch.rand((d, 12), device=dev) for d in dims]
    with pytest.raises(P.MttkrpError) as e:
        h.mttkrp_mode(0, fac)
    assert e.value.status == 3          # rank 12 unsupported
    h.destroy()


@pytest.mark.parametrize("order", ["revcyclic", "desc", "asc", "cyclic"])
@pytest.mark.parametrize("blocked", ["0", "1"])
def test_remap_walks_and_key_orders(P, monkeypatch, order, blocked):
    # Every key-order policy and both remap walks (destination order / source-block order, with blocks
    # small enough that the tensor spans many of them) obey the same contract: the permutation equals the
    # oracle's stable sort by the reported key tuple, the remapped copy is that sorted COO, Y within tolerance.
    monkeypatch.setenv("MTTKRP_KEY_ORDER", order)
    monkeypatch.setenv("MTTKRP_REMAP_BLOCKED", blocked)
    monkeypatch.setenv("MTTKRP_REMAP_BLOCK_LOG2", "12")
    for cfg, nnz, R in [(1, 150_001, 32), (3, 90_007, 16), (4, 60_013, 8)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        N = len(spec.dims)
        worst, info = _run_case(P, spec.dims, t.idx, t.vals, R, seed=6, order_modes=list(range(N)) + [0, N - 1, 1])
        assert info["remap_blocked"] == [int(blocked)] * N
        if order == "revcyclic":
            assert info["key_order"] == [[(d - j) % N for j in range(N)] for d in range(N)]


@pytest.mark.parametrize("order", ["revcyclic", "desc"])
def test_two_pass_remap(P, monkeypatch, order):
    # The third walk of Alg. 3: records first grouped by destination window (scatter, sequential reads), then gathered
    # inside the window.  Same contract as the other walks: permutation, remapped copy and Y equal the oracle's.
    monkeypatch.setenv("MTTKRP_KEY_ORDER", order)
    monkeypatch.setenv("MTTKRP_REMAP_TWOPASS", "1")
    monkeypatch.setenv("MTTKRP_TWOPASS_WINDOW_LOG2", "11")          # many windows even at test sizes
    for cfg, nnz, R in [(1, 150_001, 32), (2, 260_003, 32), (3, 90_007, 16), (4, 60_013, 8)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        N = len(spec.dims)
        worst, info = _run_case(P, spec.dims, t.idx, t.vals, R, seed=6, order_modes=list(range(N)) + [0, N - 1, 1, 2, 0])
        assert 2 in info["remap_blocked"] and info["remaps_done"] == 0
        assert all(w == 2 or w == 1 for w in info["remap_blocked"])


@pytest.mark.parametrize("pack", ["0", "1"])
def test_record_formats_for_four_and_more_modes(P, monkeypatch, pack):
    # N >= 4: packed 16-byte records (bit-level layout) and the 4*(N+1)-byte fallback
    # compute the same thing; both remap walks; record_bytes reports the format.
    monkeypatch.setenv("MTTKRP_PACK", pack)
    monkeypatch.setenv("MTTKRP_REMAP_BLOCK_LOG2", "12")
    for dims, nnz, R in [((37, 50, 19, 64), 20_011, 32), ((9, 30, 1000, 7, 24), 30_013, 16),
                         ((5, 4, 6, 3, 4, 5), 3_001, 8), ((3, 2, 4, 2, 3, 2, 5, 2), 2_003, 64),
                         ((3, 2, 4, 2, 3, 2, 5, 2), 2_003, 8)]:     # unpacked: > 48 KB of shared memory per block
        spec = W.TensorSpec("fmt", list(dims), nnz, [1.1] + [0.0] * (len(dims) - 1), "uniform", (R,), 91)
        t = W.generate_tensor(spec)
        N = len(dims)
        worst, info = _run_case(P, list(dims), t.idx, t.vals, R, seed=8, order_modes=list(range(N)) + [1, 0])
        assert info["record_bytes"] == (16 if pack == "1" else 4 * (N + 1))


@pytest.mark.parametrize("pack", ["0", "1"])
@pytest.mark.parametrize("dims,cid", [((400_000, 30, 17, 2500, 9, 12), 96), ((300_000, 6, 5, 700, 4, 3, 40, 2), 98)])
def test_mid_size_six_and_eight_modes_all_entries(P, monkeypatch, dims, cid, pack):
    # More than 4 modes is one of the paper's claims (Sec. 5.6), and the N = 6..8 instantiations have
    # their own occupancy targets and > 48 KB shared-memory geometry.  A million nonzeros gives them what the tiny
    # tensors cannot: hundreds of shards (a multi-wave grid), rows split across many shards (the 2..40-row modes),
    # empty rows (the Zipf mode), both record formats, the narrowest and the widest rank - every entry of every Y_d and
    # every permutation against the oracle.
    monkeypatch.setenv("MTTKRP_PACK", pack)
    N = len(dims)
    spec = W.TensorSpec(f"mid{N}", list(dims), 1_000_003, [1.2] + [0.0] * (N - 1), "uniform", (8, 64), cid)
    t = W.generate_tensor(spec)
    for R in (8, 64):
        worst, info = _run_case(P, list(dims), t.idx, t.vals, R, seed=cid + R, check_perm=(R == 8))
        assert info["record_bytes"] == (16 if pack == "1" else 4 * (N + 1))
        assert info["num_shards"] >= 100
        assert max(info["num_split_rows"]) > 0 and info["num_empty_rows"][0] > 0


def test_wide_index_tensor_falls_back_to_unpacked_records(P):
    # 3 x 22 bits of leading keys do not fit the 64-bit key string: the handle keeps 20-byte records.
    # (The cell count exceeds 64 bits, so the COO list is drawn directly; duplicates are legal and add.)
    dims = [1 << 22, 1 << 22, 1 << 22, 1 << 10]
    g = torch.Generator().manual_seed(92)
    nnz = 50_021
    idx = torch.stack([torch.randint(0, d, (nnz,), generator=g, dtype=torch.int64) for d in dims]).to(torch.int32)
    vals = torch.rand(nnz, generator=g, dtype=torch.float32)
    t = W.SparseTensor(W.TensorSpec("wide", dims, nnz, [0.0] * 4, "uniform", (8,), 92), idx, vals)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(dims, t.idx.to(dev), t.vals.to(dev))
    assert h.info()["record_bytes"] == 20
    fac_np = [np.random.default_rng(m).uniform(-1, 1, size=(d, 8)).astype(np.float32) for m, d in enumerate(dims)]
    fac = [torch.from_numpy(f).to(dev) for f in fac_np]
    rng = np.random.default_rng(5)
    for d in [0, 3]:
        Y = h.mttkrp_mode(d, fac)
        rows = np.unique(t.idx[d].numpy()[rng.choice(t.nnz, 64, replace=False)]).astype(np.int64)
        Yo, So = oracle.mttkrp_rows(dims, t.idx.numpy(), t.vals.numpy(), fac_np, d, rows)
        err, zeros_ok = oracle.normalised_error(Y[torch.from_numpy(rows).to(dev)].cpu().numpy(), Yo, So)
        assert zeros_ok and err <= TOL
    h.destroy()


def test_blocked_walk_is_chosen_from_measured_runs(P):
    # Without overrides mttkrp_create measures the runs of both walks: small modes (long runs) -> blocked.
    spec = W.CONFIGS[1].scaled(3_000_017)          # > 2 blocks of 2^20 records
    t = W.generate_tensor(spec)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
    info = h.info()
    assert info["remap_blocked"] == [1, 1, 1] and min(info["remap_avg_run"]) >= 4
    h.destroy()


@pytest.mark.parametrize("walk", ["measured", "twopass", "blocked"])
def test_workspace_beyond_bytes_held_is_the_callers(P, monkeypatch, walk):
    # info.bytes_held is a promise: after create the handle lives in workspace[0, bytes_held) - the walk maps of
    # transitions that ended up with the plain walk, and the create-time scratch, are given back.  Overwrite
    # everything from bytes_held on and every call must still match the oracle (permutation, remapped copy, Y).
    if walk == "twopass":
        monkeypatch.setenv("MTTKRP_REMAP_TWOPASS", "1")
        monkeypatch.setenv("MTTKRP_TWOPASS_WINDOW_LOG2", "11")
    if walk == "blocked":
        monkeypatch.setenv("MTTKRP_REMAP_BLOCKED", "1")
        monkeypatch.setenv("MTTKRP_REMAP_BLOCK_LOG2", "12")
    dev = torch.device("cuda:0")
    for cfg, nnz, R in [(0, 100_000, 16), (2, 260_003, 32), (3, 90_007, 8)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        dims, N = list(spec.dims), len(spec.dims)
        h = P.Mttkrp(dims, t.idx.to(dev), t.vals.to(dev))
        info = h.info()
        total = P.mttkrp_workspace_bytes(dims, t.nnz)
        held = info["bytes_held"]
        slot = -(-4 * t.nnz // 256) * 256                               # one walk map, 256-byte aligned
        users = sum(1 for w in info["remap_blocked"] if w != 0)
        assert 0 < held <= total
        if users == 0:
            assert held <= total - 2 * N * slot                         # plain walks everywhere: the whole pool is free
        else:
            assert held == total - 2 * (N - users) * slot
        if walk == "measured":
            assert users == 0                                           # too small for the blocked / two-pass walks
        else:
            assert users > 0
        off = h._ws_ptr - h.workspace.data_ptr()
        h.workspace[off + held:].fill_(0xA5)
        idx_np, vals_np = t.idx.numpy(), t.vals.numpy()
        fac_np = [np.random.default_rng(40 + m).uniform(-1, 1, size=(d, R)).astype(np.float32) for m, d in enumerate(dims)]
        fac = [torch.from_numpy(f).to(dev) for f in fac_np]
        for d in list(range(N)) + [0, N - 1, 1, 0]:                     # cyclic sweep, then out-of-order jumps
            perm = oracle.sort_perm(dims, idx_np, info["key_order"][d])
            out = torch.full((dims[d], R), float("nan"), dtype=torch.float32, device=dev)
            Y = h.mttkrp_mode(d, fac, out=out).cpu().numpy()
            gi, gv = h.export_coo()
            np.testing.assert_array_equal(gi.cpu().numpy(), idx_np[:, perm])
            np.testing.assert_array_equal(gv.cpu().numpy(), vals_np[perm])
            np.testing.assert_array_equal(h.get_perm(d).cpu().numpy().astype(np.int64), perm)
            Yo, So = oracle.mttkrp_mode(dims, idx_np, vals_np, fac_np, d, perm=perm)
            err, zeros_ok = oracle.normalised_error(Y, Yo, So)
            assert zeros_ok and err <= TOL
        assert bool((h.workspace[off + held:] == 0xA5).all()), "the handle wrote beyond bytes_held"
        h.destroy()


@pytest.mark.parametrize("variant", ["default", "deep", "unpacked", "twopass", "blocked", "fused", "alg1"])
def test_repeated_sweeps_are_bit_identical(P, monkeypatch, variant):
    # compute-sanitizer is closed on the GPU pool this library is developed on (profiles/r3_sanitizer_summary.md), so
    # racecheck cannot vouch for the shared-memory protocol of k_mttkrp (record ring aliased with the groups' partial
    # rows, __syncwarp hand-offs) or of k_scatter16 (shared atomics + one-warp scan).  What can be checked without
    # it: every reduction in the path has a FIXED order, so a sweep must reproduce itself bit for bit; a hazard between
    # warps or lanes shows up as a run-to-run difference in some entry or some record.  12 sweeps per tensor, every
    # kernel variant, outputs and the resident copy compared with the first sweep's (which _run_case-style tests
    # elsewhere compare with the oracle), NaN-poisoned outputs each time.
    env = {"deep": {"MTTKRP_FORCE_DEEP": "1"}, "unpacked": {"MTTKRP_PACK": "0"},
           "twopass": {"MTTKRP_REMAP_TWOPASS": "1", "MTTKRP_TWOPASS_WINDOW_LOG2": "11"},
           "blocked": {"MTTKRP_REMAP_BLOCKED": "1", "MTTKRP_REMAP_BLOCK_LOG2": "12"},
           "fused": {"MTTKRP_FUSE": "1"}, "alg1": {"MTTKRP_SHARD_POLICY": "alg1", "MTTKRP_KAPPA": "37"}}.get(variant, {})
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    dev = torch.device("cuda:0")
    for cfg, nnz, R in [(1, 400_009, 32), (2, 300_011, 64), (3, 250_007, 32), (4, 200_003, 16)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        N = len(spec.dims)
        h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
        fac = [f.to(dev) for f in W.generate_factors(spec, R)]
        ref, ref_coo = None, None
        for rep in range(12):
            outs = [torch.full((d, R), float("nan"), dtype=torch.float32, device=dev) for d in spec.dims]
            h.mttkrp_sweep(fac, outs)
            coo = h.export_coo()                                          # layout N-1 after a sweep
            if ref is None:
                ref, ref_coo = outs, coo
                assert all(bool(torch.isfinite(y).all()) for y in outs)
                continue
            for d in range(N):
                assert torch.equal(outs[d], ref[d]), f"{variant} cfg{cfg} sweep {rep} mode {d} differs from sweep 0"
            assert torch.equal(coo[0], ref_coo[0]) and torch.equal(coo[1], ref_coo[1])
        h.destroy()


def _sample_rows(idx_d, dim, rng, k=48):
    """Heaviest rows, rows around shard boundaries' worth of mass, and random rows."""
    counts = torch.bincount(idx_d.long(), minlength=dim)
    heavy = torch.topk(counts, min(8, dim)).indices.cpu().numpy()
    present = torch.nonzero(counts > 0).flatten().cpu().numpy()
    empty = torch.nonzero(counts == 0).flatten().cpu().numpy()
    pick = [heavy, rng.choice(present, size=min(k, present.size), replace=False)]
    if empty.size:
        pick.append(rng.choice(empty, size=min(4, empty.size), replace=False))
    return np.unique(np.concatenate(pick)).astype(np.int64)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_full_size_all_entries(P, cfg):
    # BASELINE.json configs[1..4] at FULL size, in the launch configuration bench.py times (mttkrp_sweep, steady
    # state, default kernel variants).  For every mode: the remap permutation equals the oracle's stable sort
    # bit-exactly (Observation 1), the remapped tensor copy is that sorted COO, and EVERY entry
    # of Y_d is compared with the fp64 oracle (rows split over all host cores) at 1e-5 normalised.
    spec = W.CONFIGS[cfg]
    R = 32
    dev = torch.device("cuda:0")
    t = W.generate_tensor(spec, dev)
    N = len(spec.dims)
    fac = W.generate_factors(spec, R, dev)
    h = P.Mttkrp(spec.dims, t.idx, t.vals)
    info = h.info()
    assert info["num_shards"] * info["shard_nnz"] >= spec.nnz > (info["num_shards"] - 1) * info["shard_nnz"]
    h.mttkrp_sweep(fac)                                   # warm-up sweep: steady state starts in layout N-1
    outs = [torch.full((spec.dims[d], R), float("nan"), dtype=torch.float32, device=dev) for d in range(N)]
    h.mttkrp_sweep(fac, outs)
    idx_np, vals_np = t.idx.cpu().numpy(), t.vals.cpu().numpy()
    fac_np = [f.cpu().numpy() for f in fac]
    threads = max(2, oracle.max_threads())
    for d in range(N):
        order = info["key_order"][d]
        assert order[0] == d and sorted(order) == list(range(N))
        perm = oracle.sort_perm(spec.dims, idx_np, order)
        perm_t = torch.from_numpy(perm).to(dev)
        assert torch.equal(h.get_perm(d).long(), perm_t), f"cfg {cfg} mode {d}: remap permutation differs from the oracle"
        h.remap_to(d)
        gi, gv = h.export_coo()
        assert torch.equal(gi, t.idx[:, perm_t]) and torch.equal(gv, t.vals[perm_t])
        del gi, gv, perm_t
        Yo, So = oracle.mttkrp_mode(spec.dims, idx_np, vals_np, fac_np, d, perm=perm, threads=threads)
        err, zeros_ok = oracle.normalised_error(outs[d].cpu().numpy(), Yo, So)
        assert zeros_ok and err <= TOL, f"cfg {cfg} mode {d}: normalised error {err:.3e}"
        del Yo, So, perm
    # cross-mode invariant on the full outputs (fp32 inputs, fp64 reduction): sum_i,r Y_d * A_d is mode-independent
    inv = [float((outs[d].double() * fac[d].double()).sum().item()) for d in range(N)]
    scale = float(sum((outs[d].double().abs() * fac[d].double().abs()).sum().item() for d in range(N)) / N)
    for d in range(1, N):
        assert abs(inv[d] - inv[0]) <= 1e-6 * scale
    h.destroy()


@pytest.mark.parametrize("R", [8, 16, 64])
def test_full_size_rank_sweep_config5(P, R):
    # BASELINE.json configs[4] (5 modes, 60M nonzeros) at the other ranks of its sweep, full size, steady state;
    # sampled output rows (heaviest, random, empty) against the oracle.  R = 32 is in test_full_size_all_entries.
    spec = W.CONFIGS[4]
    dev = torch.device("cuda:0")
    t = W.generate_tensor(spec, dev)
    N = len(spec.dims)
    fac = W.generate_factors(spec, R, dev)
    h = P.Mttkrp(spec.dims, t.idx, t.vals)
    h.mttkrp_sweep(fac)
    outs = h.mttkrp_sweep(fac)
    idx_np, vals_np = t.idx.cpu().numpy(), t.vals.cpu().numpy()
    fac_np = [f.cpu().numpy() for f in fac]
    rng = np.random.default_rng(100 + R)
    for d in range(N):
        rows = _sample_rows(t.idx[d], spec.dims[d], rng)
        Yo, So = oracle.mttkrp_rows(spec.dims, idx_np, vals_np, fac_np, d, rows)
        Y = outs[d][torch.from_numpy(rows).to(dev)].cpu().numpy()
        err, zeros_ok = oracle.normalised_error(Y, Yo, So)
        assert zeros_ok and err <= TOL, f"R {R} mode {d}: normalised error {err:.3e}"
    h.destroy()


@pytest.mark.parametrize("deep", ["0", "1"])
def test_kernel_variants_all_entries(P, monkeypatch, deep):
    # The MTTKRP kernel has two look-ahead variants for N <= 3; the library picks by the size
    # of the input factors, so the deeper one only runs on full-size configs[2] by default.  MTTKRP_FORCE_DEEP
    # pins the variant at create: both get the element-by-element comparison at sizes where every entry of every
    # Y_d is checked (tiny tensors, configs[0] at full size, the scaled shape classes of configs[1] and [2]).
    monkeypatch.setenv("MTTKRP_FORCE_DEEP", deep)
    for dims, nnz, dup in [((4, 3, 5), 30, False), ((5, 4), 12, True), ((7, 1, 3), 15, False)]:
        t = W.tiny_tensor(dims, nnz, seed=len(dims) * 100 + nnz, duplicates=dup)
        for R in (8, 32):
            _run_case(P, list(dims), t.idx, t.vals, R, seed=1)
    spec = W.CONFIGS[0]
    t = W.generate_tensor(spec)
    for R in (8, 16, 32, 64):
        _run_case(P, spec.dims, t.idx, t.vals, R, seed=2)
    for cfg, nnz in [(1, 300_137), (2, 300_137)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        worst, info = _run_case(P, spec.dims, t.idx, t.vals, 32, seed=3, order_modes=[0, 1, 2, 1, 0])
        assert max(info["num_split_rows"]) > 0


@pytest.mark.parametrize("keep", ["0", "7", "100"])
def test_cold_row_prefetch_marks(P, monkeypatch, keep):
    # The batch variant of the kernel requests "cold" factor rows (not among the MTTKRP_PREFETCH_ROWS most frequent
    # of their factor matrix; marks in the spare bits of the record's key words) into L2 ahead of
    # their gathers.  A small K puts marks on scaled tensors: the remapped copy must still be the oracle-sorted COO
    # bit for bit (the marks never leak into indices) and every entry of every Y_d must match; the reported counts
    # follow the documented rule (cold = degree below a threshold, at most K rows are not cold).
    monkeypatch.setenv("MTTKRP_FORCE_DEEP", "1")
    monkeypatch.setenv("MTTKRP_PREFETCH_ROWS", keep)
    for dims, nnz in [((40, 30, 50), 3000), ((90, 70), 2500)]:
        t = W.tiny_tensor(dims, nnz, seed=nnz)
        for R in (8, 16, 32, 64):
            _run_case(P, list(dims), t.idx, t.vals, R, seed=5)
    spec = W.CONFIGS[2].scaled(300_137)
    t = W.generate_tensor(spec)
    worst, info = _run_case(P, spec.dims, t.idx, t.vals, 32, seed=6, order_modes=[0, 1, 2, 0, 2, 1])
    K = int(keep)
    for m in range(3):
        deg = np.bincount(t.idx[m].numpy(), minlength=spec.dims[m])
        if K == 0:
            assert info["cold_rows"][m] == 0 and info["cold_degree"][m] == 0
        else:
            T = info["cold_degree"][m]
            assert info["cold_rows"][m] == int((deg < T).sum())
            assert spec.dims[m] - info["cold_rows"][m] <= K


def test_calls_on_different_streams_are_ordered(P):
    # Calls on one handle share the tensor copies and the carry buffer.  The library orders them itself: a call
    # on another stream waits for the handle's previous work (include/mttkrp.h conventions), so issuing the modes
    # round-robin on three streams with no synchronisation in between gives the single-stream results bit for bit.
    spec = W.CONFIGS[1].scaled(2_000_003)
    t = W.generate_tensor(spec)
    dev = torch.device("cuda:0")
    R = 32
    fac = [f.to(dev) for f in W.generate_factors(spec, R)]
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
    ref = [y.clone() for y in h.mttkrp_sweep(fac)]
    streams = [torch.cuda.Stream() for _ in range(3)]
    outs = [[torch.empty_like(ref[d]) for d in range(3)] for _ in range(4)]
    torch.cuda.synchronize()
    k = 0
    for rep in range(4):
        for d in (0, 1, 2):
            with torch.cuda.stream(streams[k % 3]):
                h.mttkrp_mode(d, fac, out=outs[rep][d])
            k += 2                                       # consecutive calls never share a stream
    torch.cuda.synchronize()
    for rep in range(4):
        for d in range(3):
            assert torch.equal(outs[rep][d], ref[d])
    h.destroy()


def test_out_of_order_calls_use_one_composed_pass(P):
    # Any d in any order: a jump over k layouts composes the stored position maps and moves the records ONCE
    # (SURVEY.md Sec. 8(a) state machine); the resident copy must equal the oracle-sorted COO of the target layout.
    for cfg, nnz, R in [(1, 120_011, 16), (4, 90_017, 8)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        N = len(spec.dims)
        dev = torch.device("cuda:0")
        h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
        info = h.info()
        idx_np, vals_np = t.idx.numpy(), t.vals.numpy()
        seq = [2, 0, 2, 1] if N == 3 else [3, 1, 0, 4, 2, 2, 0]
        done = 0
        cur = 0
        for d in seq:
            h.remap_to(d)
            done += 1 if d != cur else 0
            cur = d
            assert h.info()["remaps_done"] == done and h.info()["cur_layout"] == d
            perm = oracle.sort_perm(spec.dims, idx_np, info["key_order"][d])
            gi, gv = h.export_coo()
            np.testing.assert_array_equal(gi.cpu().numpy(), idx_np[:, perm])
            np.testing.assert_array_equal(gv.cpu().numpy(), vals_np[perm])
        fac_np = [np.random.default_rng(m).uniform(-1, 1, size=(dd, R)).astype(np.float32) for m, dd in enumerate(spec.dims)]
        fac = [torch.from_numpy(f).to(dev) for f in fac_np]
        for d in ([1, 0] if N == 3 else [4, 1]):
            Y = h.mttkrp_mode(d, fac).cpu().numpy()
            Yo, So = oracle.mttkrp_mode(spec.dims, idx_np, vals_np, fac_np, d)
            err, zeros_ok = oracle.normalised_error(Y, Yo, So)
            assert zeros_ok and err <= TOL
        h.destroy()


def test_fused_remap_inside_the_compute_kernel(P, monkeypatch):
    # SURVEY.md Sec. 8(f) f1 / Alg. 4 lines 15-19: with MTTKRP_FUSE=1 the MTTKRP kernel of mode d
    # also executes Alg. 3 (T_out[remap id for mode (d+1) mod N] = record), so the next mode only swaps the copies.
    # Same bars as the separate pass: the resident copy after every call is the oracle-sorted COO (bit-exact), Y
    # within tolerance; out-of-order calls fall back to the composed gather pass.
    monkeypatch.setenv("MTTKRP_FUSE", "1")
    monkeypatch.setenv("MTTKRP_REMAP_BLOCK_LOG2", "12")
    for cfg, nnz, R in [(1, 150_011, 32), (2, 120_007, 32), (3, 90_013, 16), (4, 70_001, 8), (0, 100_000, 16)]:
        spec = W.CONFIGS[cfg].scaled(nnz)
        t = W.generate_tensor(spec)
        N = len(spec.dims)
        worst, info = _run_case(P, spec.dims, t.idx, t.vals, R, seed=11, order_modes=list(range(N)) * 2 + [1, 0, N - 1, 0, 1])
        assert info["fused_remap"] is True
    # a full cyclic sweep costs no separate record pass: N swaps
    spec = W.CONFIGS[1].scaled(200_003)
    t = W.generate_tensor(spec)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
    fac = [f.to(dev) for f in W.generate_factors(spec, 32)]
    ref = None
    for rep in range(3):
        h.timing_begin()
        outs = h.mttkrp_sweep(fac)
        tm = h.timing_end()
        assert tm["mttkrp_launches"] == 3
        if ref is None:
            ref = [y.clone() for y in outs]
        for d in range(3):
            assert torch.equal(outs[d], ref[d])
    assert h.info()["remaps_done"] == 8                    # 0->1->2 in the first sweep, then 3 per sweep: all swaps
    h.destroy()
