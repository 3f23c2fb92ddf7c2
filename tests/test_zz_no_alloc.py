"""chfpe_spectrum_2d_static: the entry point that allocates nothing (its scratch is a static device array inside the
library, for callers under CUDA graph capture or in harnesses that forbid cudaMalloc).  Collected last on purpose
(the suite runs with pytest -x).  Compares it with the existing chfpe_spectrum_2d path on two calls in a row --
the second with other sizes, so that what the first left in the shared scratch would show -- and checks the size limit.
Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def test_static_scratch_spectrum_matches_the_existing_path_twice_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2509_25840_b200 as P
    rng = np.random.default_rng(23)
    dev = torch.device("cuda", 0)
    # first the full delay grid of BASELINE configs[4] (64 x 256), then a smaller ragged case
    for (n1, n2, nw1, nw2, s1, s2) in ((64, 256, 37, 65, -1, -1), (19, 33, 7, 11, -1, 1)):
        R = rng.standard_normal((n1, n2))
        om1, om2 = np.linspace(0.0, 3.0, nw1), np.linspace(-2.0, 2.5, nw2)
        ref = P.spectrum_2d(R, 0.02, 0.015, om1, om2, s1, s2)          # existing path: caller-provided scratch
        Rd = torch.from_numpy(R).to(dev)
        o1, o2 = torch.from_numpy(om1).to(dev), torch.from_numpy(om2).to(dev)
        out = torch.full((nw1, nw2), float("nan"), dtype=torch.float64, device=dev)
        free0 = torch.cuda.mem_get_info()[0]
        P.spectrum_2d_static_device(Rd, 0.02, 0.015, o1, o2, out, s1, s2)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0                   # nothing was allocated on the device
        got = out.cpu().numpy()
        scale = np.max(np.abs(ref))
        assert np.max(np.abs(got - ref)) <= 1e-12 * scale              # tolerance of tests/test_gpu_spectra.py
        assert np.array_equal(got, ref)                                # same kernels, same order: bit-identical


def test_static_scratch_spectrum_rejects_sizes_beyond_its_maximum():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2509_25840_b200 as P
    dev = torch.device("cuda", 0)
    n1, nw2 = 257, 256                                                  # 257 * 256 = 65792 > 65536
    assert n1 * nw2 > P.SPECTRUM_STATIC_MAX
    Rd = torch.zeros((n1, 4), dtype=torch.float64, device=dev)
    o1 = torch.zeros(3, dtype=torch.float64, device=dev)
    o2 = torch.zeros(nw2, dtype=torch.float64, device=dev)
    out = torch.zeros((3, nw2), dtype=torch.float64, device=dev)
    with pytest.raises(P.ChfpeError, match="-2"):                       # CHFPE_ERR_WORKSPACE
        P.spectrum_2d_static_device(Rd, 0.1, 0.1, o1, o2, out)
    ok = torch.zeros((256, 4), dtype=torch.float64, device=dev)         # 256 * 256 = the maximum itself is accepted
    P.spectrum_2d_static_device(ok, 0.1, 0.1, o1, o2, out)
    torch.cuda.synchronize()
