"""Pin of the all-cores oracle variant (oracle/vmat_oracle_mt.c, timed by bench.py's cpu_baseline second leg) against
the plain single-thread oracle: same functions on shares of the input, so every output agrees to 1e-12 relative
(FP64 additions in another order) and the selection bit for bit."""
import numpy as np
import pytest

import oracle
import synth
from conftest import as_np


@pytest.mark.parametrize("n_threads", [1, 2, 3, 7, 16])
@pytest.mark.parametrize("scale", [1.0, 14.0])
def test_threaded_evaluation_equals_the_plain_one(cfg0, n_threads, scale):
    A = as_np(cfg0)
    x = synth.draw_x(A["n_b"], 5, scale=scale).numpy()
    args = (A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x, A["sid"], A["T"], A["wo"], A["wu"], A["lco"], A["aro"])
    ref = oracle.price_eval(*args)
    got = oracle.price_eval_mt(*args, n_threads=n_threads)
    for name in ("d", "g", "p"):
        r, v = getattr(ref, name), getattr(got, name)
        assert np.abs(v - r).max() <= 1e-12 * max(1.0, np.abs(r).max()), name
    assert abs(got.F - ref.F) <= 1e-12 * abs(ref.F)
    if np.array_equal(got.p_f32, ref.p_f32):                      # same FP32 prices -> the same selection, bit for bit
        assert np.array_equal(got.L, ref.L) and np.array_equal(got.R, ref.R)
        assert np.array_equal(got.row_price, ref.row_price) and np.array_equal(got.angle_price, ref.angle_price)
    assert got.best_angle == ref.best_angle


def test_threaded_selection_is_bit_identical(cfg0):
    A = as_np(cfg0)
    rng = np.random.default_rng(4)
    p = rng.integers(-4, 5, A["n_b"]).astype(np.float32)
    L, R, rp = oracle.select_rows(p, A["lco"])
    lib = oracle._load_mt()
    for nt in (1, 5, 64, 200):                                    # more threads than rows: empty shares
        n_rows = A["lco"].size - 1
        L2, R2, rp2 = np.zeros(n_rows, np.int32), np.zeros(n_rows, np.int32), np.zeros(n_rows, np.float64)
        lco = np.ascontiguousarray(A["lco"], np.int32)
        lib.oracle_mt_select_rows(nt, n_rows, lco.ctypes.data, p.ctypes.data, L2.ctypes.data, R2.ctypes.data,
                                  rp2.ctypes.data, int(np.diff(lco).max()))
        assert np.array_equal(L, L2) and np.array_equal(R, R2) and np.array_equal(rp, rp2)


def test_more_threads_than_triplets():
    vox = np.array([0, 1], np.int32); beam = np.array([1, 0], np.int32); val = np.array([2.0, 3.0], np.float32)
    x = np.array([1.0, 10.0], np.float32)
    args = (vox, beam, val, 2, 2, x, np.zeros(2, np.uint8), np.array([5.0], np.float32), np.array([1.0], np.float32),
            np.array([1.0], np.float32), np.array([0, 2], np.int32), np.array([0, 1], np.int32))
    ref, got = oracle.price_eval(*args), oracle.price_eval_mt(*args, n_threads=8)
    assert np.array_equal(ref.d, got.d) and np.array_equal(ref.p, got.p) and ref.F == got.F
