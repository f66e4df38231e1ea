"""lb_diagnostics_noalloc (include/lb.h): the diagnostics with their scratch in a static __device__ array, against the
existing lb_get_diagnostics on the same states.  Collected last on purpose (pytest -x: a failure here hides nothing)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
from paper_2112_08264_b200 import binding as B
from paper_2112_08264_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype,tol_m,tol_p", [(B.LB_F64, 1e-13, 1e-10), (B.LB_F32, 1e-5, 1e-3)])
def test_noalloc_diagnostics_match_existing_path_on_two_calls_in_a_row(dtype, tol_m, tol_p):
    if not torch.cuda.is_available():
        pytest.skip("no GPU")
    stream = torch.cuda.Stream()
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    # a larger box first, so that the second call finds the first one's partials beyond its own in the shared array
    big, cfg = w.CONFIGS[1], w.CONFIGS[0]
    for c_, steps in ((big, 2), (cfg, 3)):
        rr, rb = c_.fields()
        mask = None
        if c_ is cfg:                                            # second call: with solid nodes too (the links path)
            mask = np.zeros(c_.n_nodes, dtype=np.uint8)
            mask[:: 37] = 1
        with B.Box(c_.nx, c_.ny, c_.nz, 0.8, 1.3, 0.9, dtype=dtype, cuda_stream=stream.cuda_stream) as box:
            if mask is not None:
                box.set_solid_mask(mask)
            box.set_fields(rr, rb)
            for call in range(2):                                # two calls in a row on this context, the state stepped in between
                box.step(steps)
                out.fill_(float("nan"))
                torch.cuda.synchronize()
                l0 = box.launch_count()
                box.diagnostics_noalloc(out.data_ptr())
                assert box.launch_count() - l0 == 2
                box.sync()
                got = out.cpu().numpy()
                m, p = box.get_diagnostics()                     # the existing path, same state
                assert np.all(np.isfinite(got))
                assert np.abs(got[:2] / m - 1).max() < tol_m, (got, m)
                assert np.abs(got[2:] - p).max() < tol_p, (got, p)


def test_noalloc_rejects_bad_arguments():
    if not torch.cuda.is_available():
        pytest.skip("no GPU")
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    with B.Box(32, 32, 32, 1.0, 1.0, 1.2) as box:
        with pytest.raises(B.LBError):
            box.diagnostics_noalloc(out.data_ptr())              # LB_ESTATE: no fields yet
        rr, rb = w.CONFIGS[0].fields()
        box.set_fields(rr, rb)
        with pytest.raises(B.LBError):
            box.diagnostics_noalloc(0)                           # NULL output


def test_noalloc_rejects_a_box_beyond_the_static_scratch():
    """2^28 nodes is the limit (16384 partials of 16384 nodes): a 1024 x 1024 x 257 fp32 box (88 GB of state) is one plane beyond it."""
    if not torch.cuda.is_available():
        pytest.skip("no GPU")
    if torch.cuda.mem_get_info()[0] < 100e9:
        pytest.skip("not enough free device memory for a box beyond 2^28 nodes")
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    with B.Box(1024, 1024, 257, 1.0, 1.0, 1.2, dtype=B.LB_F32) as box:
        with pytest.raises(B.LBError, match="2\\^28"):
            box.diagnostics_noalloc(out.data_ptr())
