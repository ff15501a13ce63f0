"""gmmnlse_overlap_tensor_noalloc: the Eq. 2 Gram product with its scratch in a static device array (no cudaMalloc),
against the existing gmmnlse_overlap_tensor, on calls in a row that share that array.

Named test_zz_* so that pytest collects it last (the suite runs with pytest -x).  Passes alone in a fresh process and
after the other tests: it depends on nothing but the library and uses its own inputs.
"""
import numpy as np
import pytest

from oracle import gmmnlse_oracle as O
from paper_1708_05324_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1708_05324_b200 import binding
    binding.load_library()
    return binding


def _noalloc(B, F, dA, stream=None):
    Fd = torch.from_numpy(np.ascontiguousarray(F, dtype=np.float64)).cuda()
    P = F.shape[0]
    Sd = torch.full((P, P, P, P), float("nan"), dtype=torch.float64, device="cuda")
    B.overlap_tensor_noalloc(Fd, dA, Sd, stream)
    torch.cuda.synchronize()
    return Sd.cpu().numpy()


def test_noalloc_matches_existing_path_on_calls_in_a_row(B):
    """Three calls back to back on the one shared scratch array -- 6 GRIN modes on a 64 x 64 grid (the limits), then a
    smaller problem (3 modes, 32 x 32: stale contents of the larger call stay in the array around it), then the first
    again -- each against the existing path at the tolerance of test_overlap_tensor_gpu_vs_oracle (2e-6 of the
    largest entry), and the first against the oracle's Eq. 2."""
    lim = B.overlap_tensor_noalloc_limits()
    assert lim["P_max"] == 6 and lim["G_max"] == 4096 and 4 << 20 < lim["scratch_bytes"] < 6 << 20
    F6, dA6, _ = W.grin_modes(2, n_grid=64)
    F3, dA3, _ = W.grin_modes(1, n_grid=32)
    assert F6.shape[0] == 6 and F3.shape[0] == 3
    first = None
    for F, dA in ((F6, dA6), (F3, dA3), (F6, dA6)):
        ref = B.overlap_tensor(F, dA)                              # existing path: per-call cudaMalloc scratch
        got = _noalloc(B, F, dA)
        assert got.shape == ref.shape and np.isfinite(got).all()
        assert np.abs(got - ref).max() <= 2e-6 * np.abs(ref).max()
        if first is None:
            first = got
            assert np.abs(got - O.overlap_tensor(F, dA)).max() <= 2e-6 * np.abs(ref).max()
    assert np.array_equal(got, first)                              # same input, same bits: nothing leaks between calls


def test_noalloc_on_a_user_stream_and_unnormalised_input(B):
    F6, dA6, _ = W.grin_modes(2, n_grid=64)
    ref = B.overlap_tensor(F6, dA6)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        got = _noalloc(B, 1e3 * F6, dA6, st)                       # Eq. 2 is scale-invariant in F
    assert np.abs(got - ref).max() <= 2e-6 * np.abs(ref).max()


def test_noalloc_rejects_sizes_beyond_the_static_scratch(B):
    Sd = torch.zeros((7, 7, 7, 7), dtype=torch.float64, device="cuda")
    for shape in ((7, 1024), (2, 8192), (2, 48)):                  # too many modes; too many grid points; G % 32 != 0
        Fd = torch.ones(shape, dtype=torch.float64, device="cuda")
        with pytest.raises(B.GmmnlseError) as e:
            B.overlap_tensor_noalloc(Fd, 1.0, Sd)
        assert e.value.status == B.EUNSUPPORTED
        assert "gmmnlse_overlap_tensor_noalloc" in str(e.value)
    with pytest.raises(B.GmmnlseError) as e:
        B.overlap_tensor_noalloc(torch.ones((2, 64), dtype=torch.float64, device="cuda"), 0.0, Sd)
    assert e.value.status == B.EINVAL
