"""The seeded input generators: numpy and torch versions agree; values are a function of the
global linear index only; the workload table matches BASELINE.json's sizes."""
import numpy as np
import torch

from paper_2211_05322_b200 import inputs


def test_mix64_known_values():
    # splitmix64 finaliser: mix(0) = 0 and a bijection on a sample
    x = np.arange(0, 1 << 16, dtype=np.uint64)
    y = inputs.mix64_np(x)
    assert y[0] == 0
    assert len(np.unique(y)) == len(x)


def test_numpy_and_torch_generators_agree():
    for name in ("c1", "c1i"):
        w = inputs.CONFIGS[name]
        a = inputs.global_tensor(w)
        b = inputs.global_tensor_torch(w, "cpu").numpy()
        assert a.dtype == b.dtype and np.array_equal(a, b)
        assert np.array_equal(a.reshape(-1), np.arange(a.size, dtype=np.float32))
    w = inputs.CONFIGS["c3"]._replace(shape=(2, 5, 8, 8))
    a = inputs.global_tensor(w, chunk=100)
    b = inputs.global_tensor_torch(w, "cpu", chunk=77).numpy()
    assert a.dtype == np.int16 and np.array_equal(a, b)
    assert len(np.unique(a)) > a.size // 2           # not degenerate
    for dt in ("u8", "i32", "i64"):
        w2 = w._replace(dtype=dt)
        assert np.array_equal(inputs.global_tensor(w2), inputs.global_tensor_torch(w2, "cpu").numpy())


def test_workload_sizes():
    nbytes = lambda w: int(np.prod(w.shape)) * inputs.elem_bytes(w.dtype)
    assert nbytes(inputs.CONFIGS["c1"]) == 512
    assert nbytes(inputs.CONFIGS["c2"]) == 128 << 20
    assert nbytes(inputs.CONFIGS["c3"]) == 20 << 20
    assert nbytes(inputs.CONFIGS["c4"]) == 1536 << 20
    for nb in inputs.SWEEP_BYTES:
        w = inputs.sweep_workload("P1", "m8", nb)
        assert nbytes(w) == nb and w.shape[2] == 4096
    assert inputs.sweep_workload("P5", "m4", 1 << 30).shape == (64, 2048, 4096)
    assert nbytes(inputs.table2_workload(4)) == 1 << 30
    assert inputs.get_workload("sweep_P2_m4_256MiB").src_mesh == (1, 4)
    assert inputs.get_workload("t2_8").dst_mesh == (3, 2)
