"""Pins of the C data oracle (oracle/reshard_oracle.c) to things other than itself.

Each test is chosen so that a plausible mistake in the oracle (wrong device numbering,
S^{01} axis order swapped, a transposed mesh, lo/hi off by one shard, source replica chosen
wrongly, dims iterated in the wrong order) fails at least one of them.
"""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

from oracle import data_oracle as do
import golden_io


# ---------------------------------------------------------------- paper's worked example

def test_fig2_spec2_devices_4_and_5_hold_elements_0_to_7():
    """values printed by the paper."""
    g = golden_io.load("fig2_example.txt")
    D = np.array(g["matrix_values"], dtype=np.float32).reshape(g["matrix_shape"])
    for dev, key in ((4, "spec2_device4_elements"), (5, "spec2_device5_elements")):
        local = dev - g["mesh_b_devices"][0]
        sh = do.shard_from_global(D, g["mesh_b"], g["spec2"], local)
        assert sh.reshape(-1).tolist() == g[key]
    # devices 6, 7 hold the other unique 2x4 slice
    for local in (2, 3):
        assert do.shard_from_global(D, g["mesh_b"], g["spec2"], local).reshape(-1).tolist() == list(range(8, 16))


def test_fig2_task1_and_task2_results():
    """Task 1: Spec 1 (one row per device of Mesh_A) -> Spec 2; the first unit task carries
    [0,1,2,3] to devices 4 and 5, so both must end with rows 0-1 = 0..7."""
    g = golden_io.load("fig2_example.txt")
    D = np.array(g["matrix_values"], dtype=np.int32).reshape(4, 4)
    src = [np.array([[4 * r + c for c in range(4)]], dtype=np.int32) for r in range(4)]   # row r on device r
    for r in range(4):
        assert np.array_equal(do.shard_from_global(D, g["mesh_a"], g["spec1"], r), src[r])
    dst = do.reshard((4, 4), g["mesh_a"], g["spec1"], g["mesh_b"], g["spec2"], src)
    assert dst[0].reshape(-1).tolist() == g["spec2_device4_elements"]
    assert dst[1].reshape(-1).tolist() == g["spec2_device5_elements"]
    assert dst[2].reshape(-1).tolist() == list(range(8, 16))
    assert dst[3].reshape(-1).tolist() == list(range(8, 16))
    # Task 2: Spec 2 on Mesh_B -> Spec 3 (S0,R) on Mesh_A: devices 0 and 1 get the first 2x4 slice.
    back = do.reshard((4, 4), g["mesh_b"], g["spec2"], g["mesh_a"], g["spec3"], dst)
    assert back[0].reshape(-1).tolist() == g["task2_first_slice_elements"]
    assert back[1].reshape(-1).tolist() == g["task2_first_slice_elements"]
    assert back[2].reshape(-1).tolist() == list(range(8, 16))


# ---------------------------------------------------------------- hand-written boxes (numpy slicing)

# (shape, mesh, spec, device, hand-written numpy index)  -- every box below was worked out by
# hand from PAPER.md:82-84, not computed by any code in this repo.
HAND_BOXES = [
    # (2,4) mesh ids [[0,1,2,3],[4,5,6,7]]: device 6 = coords (1,2)
    ((4, 8, 6), (2, 4), "S0,S1,R", 6, np.s_[2:4, 4:6, :]),
    ((4, 8, 6), (2, 4), "S1,R,S0", 6, np.s_[2:3, :, 3:6]),
    ((4, 8, 6), (2, 4), "R,S1,S0", 3, np.s_[:, 6:8, 0:3]),
    # S^{01}: degree 8, shard index c0*4+c1 = device id; S^{10}: index c1*2+c0
    ((4, 8, 6), (2, 4), "R,S01,R", 6, np.s_[:, 6:7, :]),
    ((4, 8, 6), (2, 4), "R,S10,R", 6, np.s_[:, 5:6, :]),      # (1,2) -> 2*2+1 = 5
    # (4,2) mesh ids [[0,1],[2,3],[4,5],[6,7]]: device 5 = coords (2,1): dim0 by axis 1 (size 2,
    # coord 1) -> rows 2:4; dim2 (8) by axis 0 (size 4, coord 2) -> 4:6
    ((4, 8, 8), (4, 2), "S1,R,S0", 5, np.s_[2:4, :, 4:6]),
]
HAND_BOXES += [
    # size-1 mesh axis behaves as R (R4): (1,4) mesh, S0 -> whole dim
    ((8, 16), (1, 2), "S0,R", 1, np.s_[:, :]),
    ((8, 16), (1, 2), "R,S1", 1, np.s_[:, 8:16]),
    ((8, 16), (1, 2), "S1,R", 1, np.s_[4:8, :]),
    # 1-D mesh
    ((6, 4), (3,), "S0,R", 2, np.s_[4:6, :]),
    # 4-D tensor on (2,2): device 3 = (1,1)
    ((2, 4, 6, 8), (2, 2), "R,S0,S1,R", 3, np.s_[:, 2:4, 3:6, :]),
    ((2, 4, 6, 8), (2, 2), "R,S0,S1,R", 2, np.s_[:, 2:4, 0:3, :]),
    ((2, 4, 6, 8), (2, 2), "R,S0,S1,R", 1, np.s_[:, 0:2, 3:6, :]),
]


@pytest.mark.parametrize("shape,mesh,spec,dev,idx", HAND_BOXES)
def test_shard_equals_numpy_slice_with_hand_written_box(shape, mesh, spec, dev, idx):
    D = np.arange(np.prod(shape), dtype=np.int64).reshape(shape)
    assert np.array_equal(do.shard_from_global(D, mesh, spec, dev), D[idx])
    lo, hi = do.device_box(shape, mesh, spec, dev)
    want = D[idx]
    assert tuple(h - l for l, h in zip(lo, hi)) == want.shape
    assert D[tuple(lo)] == want.reshape(-1)[0]


def _numpy_expected(D, mesh, spec, q):
    """dst shard by numpy slicing with the box of the *Python* plan oracle (independently written,
    itself pinned in test_plan_oracle_pins.py)."""
    from oracle import plan_oracle as po
    lo, hi = po.tile_box(D.shape, mesh, spec, q)
    box = D[tuple(slice(l, h) for l, h in zip(lo, hi))]
    lo0, hi0 = po.tile_box(D.shape, mesh, spec, 0)        # device 0's box has the padded extents (R5)
    out = np.zeros([h - l for l, h in zip(lo0, hi0)], dtype=D.dtype)
    out[tuple(slice(0, n) for n in box.shape)] = box
    return out


# ---------------------------------------------------------------- whole-task checks

CASES = [
    ((8, 16), (1, 2), "S0,R", (1, 2), "R,S0"),
    ((8, 16), (1, 2), "S1,R", (1, 2), "R,S1"),
    ((4, 8, 16), (2, 4), "S0,R,S1", (2, 4), "S0,S1,R"),
    ((4, 8, 4, 4), (1, 4), "S0,R,R,R", (2, 2), "R,S0,S1,R"),
    ((4, 8, 4, 4), (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R"),
    ((8, 16, 12), (2, 4), "S0,S1,R", (4, 2), "S1,R,S0"),
    ((8, 8, 4), (2, 4), "R,S01,R", (2, 4), "S01,R,R"),
    ((6, 6, 2), (2, 3), "RRR", (3, 2), "RRR"),
    ((12, 6), (2, 3), "S0,S1", (3, 2), "S0,S1"),          # 2-way x 3-way cuts: unequal slices
    ((8, 4), (2, 2), "S0,S1", (4,), "S0,R"),
]


@pytest.mark.parametrize("shape,sm,ss,dm,ds", CASES)
def test_reshard_equals_numpy_slicing_and_values_encode_global_index(shape, sm, ss, dm, ds):
    D = np.arange(np.prod(shape), dtype=np.int32).reshape(shape)          # value == global linear index
    src = [np.ascontiguousarray(_numpy_expected(D, sm, ss, r)) for r in range(do.num_devices(sm))]
    dst = do.reshard(shape, sm, ss, dm, ds, src)
    assert len(dst) == do.num_devices(dm)
    for q, got in enumerate(dst):
        assert np.array_equal(got, _numpy_expected(D, dm, ds, q))
    # multithreaded run is identical
    dst8 = do.reshard(shape, sm, ss, dm, ds, src, n_threads=4)
    for a, b in zip(dst, dst8):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("shape,sm,ss,dm,ds", CASES)
def test_every_destination_element_written_exactly_once(shape, sm, ss, dm, ds):
    """The oracle writes each (q, j) once by construction; check that what it wrote is a
    permutation-free image: sentinel never survives and the per-device multiset equals the box."""
    D = np.arange(1, np.prod(shape) + 1, dtype=np.int64).reshape(shape)   # never 0
    src = do.shards_from_global(D, sm, ss)
    for q in range(do.num_devices(dm)):
        out = np.zeros(do.local_shape(shape, dm, ds), dtype=np.int64)     # sentinel 0
        do.reshard_device(shape, 8, sm, ss, dm, ds, src, q, np.int64, out=out)
        assert (out != 0).all()
        assert np.array_equal(np.sort(out.reshape(-1)), np.sort(_numpy_expected(D, dm, ds, q).reshape(-1)))


@pytest.mark.parametrize("shape,sm,ss,dm,ds", CASES)
def test_a_to_b_to_a_is_identity_on_every_replica(shape, sm, ss, dm, ds):
    rng = np.random.default_rng(7)
    D = rng.integers(-2 ** 15, 2 ** 15, size=shape).astype(np.int16)
    src = do.shards_from_global(D, sm, ss)
    dst = do.reshard(shape, sm, ss, dm, ds, src)
    back = do.reshard(shape, dm, ds, sm, ss, dst)
    for a, b in zip(src, back):
        assert np.array_equal(a, b)


def test_special_cases_reduce_to_memcpy():
    rng = np.random.default_rng(3)
    shape = (8, 6, 4)
    D = rng.integers(0, 255, size=shape).astype(np.uint8)
    # same spec, same mesh shape: per-device copy (Table 2 case 1 at device level)
    src = do.shards_from_global(D, (2, 4), "S0RR")
    dst = do.reshard(shape, (2, 4), "S0RR", (2, 4), "S0RR", src)
    for a, b in zip(src, dst):
        assert a.tobytes() == b.tobytes()
    # R..R -> R..R: every destination device gets the whole tensor (Table 2 case 8)
    src = do.shards_from_global(D, (2, 3), "RRR")
    for b in do.reshard(shape, (2, 3), "RRR", (3, 2), "RRR", src):
        assert b.tobytes() == D.tobytes()
    # 1 device -> 1 device
    dst = do.reshard(shape, (1,), "RRR", (1, 1), "RRR", [D])
    assert dst[0].tobytes() == D.tobytes()


def test_oracle_reads_lowest_index_replica():
    """R12: with deliberately different replicas the oracle's source is the lowest-index one."""
    shape = (4, 4)
    D = np.arange(16, dtype=np.int32).reshape(shape)
    src = do.shards_from_global(D, (2, 2), "S0,R")      # devices 0,1 replicas; 2,3 replicas
    src[1] = src[1] + 1000
    src[3] = src[3] + 1000
    dst = do.reshard(shape, (2, 2), "S0,R", (1, 1), "R,R", src)
    assert np.array_equal(dst[0], D)


def test_element_source_matches_full_run():
    shape, sm, ss, dm, ds = (8, 16, 12), (2, 4), "S0,S1,R", (4, 2), "S1,R,S0"
    D = np.arange(np.prod(shape), dtype=np.int64).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    dst = do.reshard(shape, sm, ss, dm, ds, src)
    rng = np.random.default_rng(0)
    for _ in range(200):
        q = int(rng.integers(0, 8))
        j = int(rng.integers(0, dst[q].size))
        dev, lin, g = do.element_source(shape, sm, ss, dm, ds, q, j)
        assert dst[q].reshape(-1)[j] == src[dev].reshape(-1)[lin] == g


def test_error_codes():
    with pytest.raises(do.OracleError) as e:
        do.local_shape((4, 4), (2, 2), "S0,S0")          # same axis twice (R3)
    assert e.value.code == do.OR_ESPEC
    with pytest.raises(do.OracleError) as e:
        do.local_shape((4, 4), (2, 2), "S2,R")           # axis out of range
    assert e.value.code == do.OR_ESPEC
    with pytest.raises(do.OracleError) as e:
        do.local_shape((4, 4), (2, 2), "S0")             # wrong length
    assert e.value.code == do.OR_ESPEC
    assert do.local_shape((5, 4), (2, 2), "S0,R") == (3, 4)   # uneven: padded extent ceil(5/2) (R5)
    assert do.local_shape((4, 8, 6), (2, 4), "RS^{01}R") == (4, 1, 6)
    assert do.local_shape((4, 8, 6), (2, 4), "(S0, S1, R)") == (2, 2, 6)


# ---------------------------------------------------------------- randomised cross-check

_SPECS2 = ["R", "S0", "S1", "S01", "S10"]


@st.composite
def _layouts(draw):
    ndim = draw(st.integers(1, 4))
    def side():
        mesh = draw(st.sampled_from([(1, 2), (2, 2), (2, 4), (4, 2), (2, 3), (3, 2), (1, 4), (4,), (3,)]))
        while True:
            spec = [draw(st.sampled_from(_SPECS2)) for _ in range(ndim)]
            axes = "".join(s[1:] for s in spec)
            if len(set(axes)) == len(axes) and all(int(a) < len(mesh) for a in axes):
                return mesh, ",".join(spec)
    sm, ss = side()
    dm, ds = side()
    shape = tuple(draw(st.sampled_from([12, 24, 7, 10, 1])) for _ in range(ndim))   # even and uneven (R5) splits
    if ndim >= 3:
        shape = tuple(min(s, 12) for s in shape)
    return shape, sm, ss, dm, ds


@settings(max_examples=60, deadline=None)
@given(_layouts())
def test_random_layouts_equal_numpy_slicing(layout):
    shape, sm, ss, dm, ds = layout
    D = np.arange(np.prod(shape), dtype=np.int32).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    for r, s in enumerate(src):
        assert np.array_equal(s, _numpy_expected(D, sm, ss, r))
    dst = do.reshard(shape, sm, ss, dm, ds, src)
    for q, got in enumerate(dst):
        assert np.array_equal(got, _numpy_expected(D, dm, ds, q))


# ---------------------------------------------------------------- uneven partitions (R5)

UNEVEN = [
    ((10,), (3,), "S0", (4,), "S0"),
    ((5, 4), (2, 2), "S0,R", (2, 2), "R,S1"),
    ((7, 9), (2, 4), "S1,S0", (4, 2), "S0,S1"),
    ((7, 5, 3), (2, 3), "S1,R,S0", (3, 2), "R,S0,S1"),
    ((2, 6), (4,), "S0,R", (2,), "S0,R"),                 # more shards than rows: devices 2, 3 hold nothing
    ((9, 10, 4), (2, 4), "S0,R,R", (3, 4), "S0,R,R"),     # Table 2 case 6 in small
    ((11, 6), (2, 4), "S01,R", (2, 3), "R,S10"),
]


def _torch_chunks(D, mesh, spec, r):
    """LIBRARY ROUTINE statement of the ceil-div convention: torch.chunk(x, k, dim) returns chunks of
    ceil(l/k) rows, the last one shorter, and FEWER than k chunks when l is small (those shards are
    empty).  Device r takes chunk p_i on every sharded dim."""
    import torch
    from oracle import plan_oracle as po
    axes = po.parse_spec(spec, D.ndim, len(mesh))
    c = po.device_coords(mesh, r)
    x = torch.from_numpy(np.ascontiguousarray(D))
    for dim, ax in enumerate(axes):
        k, p = 1, 0
        for a in ax:
            k *= mesh[a]
            p = p * mesh[a] + c[a]
        chunks = torch.chunk(x, k, dim)
        x = chunks[p] if p < len(chunks) else x.narrow(dim, 0, 0)
    return x.numpy()


@pytest.mark.parametrize("shape,sm,ss,dm,ds", UNEVEN)
def test_uneven_shards_are_torch_chunks(shape, sm, ss, dm, ds):
    D = np.arange(1, np.prod(shape) + 1, dtype=np.int32).reshape(shape)
    for mesh, spec in ((sm, ss), (dm, ds)):
        local = do.local_shape(shape, mesh, spec)
        assert local == tuple(_torch_chunks(D, mesh, spec, 0).shape)          # padded extent = first chunk
        for r in range(do.num_devices(mesh)):
            want = _torch_chunks(D, mesh, spec, r)
            lo, hi = do.device_box(shape, mesh, spec, r)
            assert tuple(h - l for l, h in zip(lo, hi)) == want.shape
            got = do.shard_from_global(D, mesh, spec, r, pad=0xEE)
            valid = tuple(slice(0, n) for n in want.shape)
            assert np.array_equal(got[valid], want)
            mask = np.ones(local, bool); mask[valid] = False
            assert (got.view(np.uint8).reshape(local + (4,))[mask] == 0xEE).all()   # padding left alone


@pytest.mark.parametrize("shape,sm,ss,dm,ds", UNEVEN)
def test_uneven_reshard_values_cover_and_identity(shape, sm, ss, dm, ds):
    D = np.arange(1, np.prod(shape) + 1, dtype=np.int64).reshape(shape)       # value = global index + 1, never 0
    src = do.shards_from_global(D, sm, ss, pad=0x77)
    dst = do.reshard(shape, sm, ss, dm, ds, src, fill=0)
    holders = np.zeros(shape, np.int32)
    for q, got in enumerate(dst):
        want = _torch_chunks(D, dm, ds, q)
        valid = tuple(slice(0, n) for n in want.shape)
        assert np.array_equal(got[valid], want)
        mask = np.ones(got.shape, bool); mask[valid] = False
        assert (got[mask] == 0).all()                                         # padding never written
        lo, hi = do.device_box(shape, dm, ds, q)
        holders[tuple(slice(l, h) for l, h in zip(lo, hi))] += 1
    assert (holders == holders.flat[0]).all() and holders.flat[0] >= 1       # every element on r_B devices
    back = do.reshard(shape, dm, ds, sm, ss, dst, fill=0x77)                  # A -> B -> A
    for a, b in zip(src, back):
        assert a.tobytes() == b.tobytes()


def test_uneven_element_source_flags_padding():
    shape, sm, ss, dm, ds = (5, 4), (2, 2), "S0,R", (2, 2), "R,S1"
    assert do.local_shape(shape, sm, ss) == (3, 4) and do.device_box(shape, sm, ss, 2) == ((3, 0), (5, 4))
    # destination device 0 holds D[:, 0:2]; its element (4, 1) comes from source device 2 (rows 3..4), local (1, 1)
    assert do.element_source(shape, sm, ss, dm, ds, 0, 4 * 2 + 1) == (2, 1 * 4 + 1, 4 * 4 + 1)
    # source side padded: shard of device 2 has 3 rows, the last one padding; as a DESTINATION it is flagged
    assert do.element_source(shape, dm, ds, sm, ss, 2, 2 * 4 + 0) == (-1, -1, -1)
