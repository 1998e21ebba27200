"""ddamg_apply_schur_noalloc: the allocation-free variant of the Schur apply (include/ddamg.h) against the
existing path.  Its scratch half spinor is a static device array inside libddamg.so, shared by every call on
the device and never cleared, so the comparison is made on two calls in a row with different inputs (the
second call finds the first call's t_o in the array), for both precisions, and the size limit is checked.
Collected last on purpose (pytest -x): a failure here hides no other test.  Runs alone in a
fresh process as well as after the rest of the suite: it creates its own contexts and inputs."""
import numpy as np
import pytest
import torch

import gen
from helpers import rel_l2

pytestmark = pytest.mark.gpu


def _dd():
    import paper_2407_08092_b200 as dd
    return dd


@pytest.mark.parametrize("prec_name,L,T", [("f32", 8, 16), ("f64", 6, 8), ("f32", 16, 32)])
def test_no_alloc_schur_apply_matches_existing_path_on_two_calls_in_a_row(prec_name, L, T):
    dd = _dd()
    f64 = prec_name == "f64"
    prec, cdt = (dd.F64, torch.complex128) if f64 else (dd.F32, torch.complex64)
    ctx = dd.Ddamg(L, T, 1.5, -0.2, 1, prec)
    ctx.load_gauge(gen.gauge_field(L, T, 1234, 0.5, True).to(cdt).cuda())
    ctx.build_clover()
    assert ctx.half_bytes <= ctx.lib.ddamg_noalloc_max_bytes()
    tol = 1e-12 if f64 else 5e-6                      # the apply tolerances of tests/test_gpu_parity.py
    y_new = ctx.half_spinor()
    for call, seed in enumerate((4321, 4322)):
        x_e, _ = ctx.pack(gen.spinor_field(L, T, seed).to(cdt).cuda())
        y_ref = ctx.apply_schur(x_e)                  # existing path: t_o in context-owned memory
        y_new.fill_(float("nan"))                     # the output must be fully written
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        ctx.apply_schur_noalloc(x_e, y_new)           # t_o in the library's static device array
        torch.cuda.synchronize()
        if call == 1:                                 # (the first call may load kernel images lazily)
            assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated inside the call"
        a = y_new.cpu().numpy().astype(np.float64)
        b = y_ref.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        assert rel_l2(a, b) <= tol, (call, rel_l2(a, b))
        assert torch.equal(y_new, y_ref)              # same kernels, same arithmetic: bit-identical
    ctx.close()


def test_no_alloc_rejects_a_lattice_beyond_the_static_scratch_and_bad_arguments():
    dd = _dd()
    ctx = dd.Ddamg(16, 48, 1.5, -0.2, 1, dd.F32)      # one half spinor = 9.4 MB > the 8 MiB array
    assert ctx.half_bytes > ctx.lib.ddamg_noalloc_max_bytes() == 8 << 20
    x, y = ctx.half_spinor(zero=True), ctx.half_spinor()
    with pytest.raises(dd.DdamgError) as e:
        ctx.apply_schur_noalloc(x, y)
    assert e.value.status == dd.EINVAL and "static scratch" in str(e.value)
    ctx.close()
    ctx = dd.Ddamg(4, 4, 1.0, -0.1, 1, dd.F32)
    x, y = ctx.half_spinor(zero=True), ctx.half_spinor()
    with pytest.raises(dd.DdamgError) as e:
        ctx.apply_schur_noalloc(x, y)                 # no gauge field yet
    assert e.value.status == dd.ESTATE
    with pytest.raises(dd.DdamgError) as e:
        ctx.apply_schur_noalloc(x, x)                 # aliasing
    assert e.value.status == dd.EINVAL
    ctx.close()
