"""GPU tests of the caller-supplied workspace (ocn_model_desc.workspace, ocn_model_workspace_bytes): a model
that lives in a torch tensor steps to the same bits as one the library allocated, and creating it allocates nothing."""
import numpy as np
import pytest
import torch

from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W

pytestmark = pytest.mark.gpu
FIELDS = ("u", "v", "w", "eta", "T", "S")


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def _torch_workspace(nbytes):
    t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda")
    return t, t.data_ptr()


def _workload(prec, ri):
    wl = W.config2(nx=96, ny=48, nz=12, steps=6, precision=prec)
    if ri:
        W.with_ri_closure(wl)
    return wl


@pytest.mark.parametrize("prec,ri", [(32, 0), (32, 1), (64, 1)])
def test_a_model_in_a_workspace_steps_to_the_same_bits(prec, ri):
    wl = _workload(prec, ri)
    a = ocn.Model(wl)
    b = ocn.Model(wl, workspace=_torch_workspace)
    assert b.info()["device_bytes"] <= b.workspace_bytes()
    a.time_step(6); b.time_step(6)
    fa, fb = a.get_fields(), b.get_fields()
    for k in FIELDS:
        assert np.array_equal(fa[k], fb[k]), (prec, ri, k)
    if ri:
        ma, mb = a.mixing(), b.mixing()                    # its output array is the library's, also for a model in a workspace
        assert np.array_equal(ma["nu"], mb["nu"]) and np.array_equal(ma["kappa"], mb["kappa"])
    a.close(); b.close()


def test_creating_a_model_in_a_workspace_allocates_nothing():
    wl = _workload(32, 1)
    warm = ocn.Model(wl, workspace=_torch_workspace)      # context, module and stream set-up happen here
    warm.time_step(1); warm.synchronize(); warm.close()
    torch.cuda.synchronize()
    holder = {}

    def ws(n):
        holder["t"] = torch.empty(int(n), dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        holder["free"] = torch.cuda.mem_get_info()[0]
        return holder["t"], holder["t"].data_ptr()

    m = ocn.Model(wl, workspace=ws)
    m.time_step(3); m.synchronize()
    assert torch.cuda.mem_get_info()[0] == holder["free"]  # not one byte of device memory besides the workspace
    m.close()


def test_workspace_is_checked():
    wl = _workload(32, 0)
    with pytest.raises(RuntimeError, match="workspace too small"):
        ocn.Model(wl, workspace=lambda n: _torch_workspace(n // 2) + (n // 2,))
    with pytest.raises(RuntimeError, match="256-byte aligned"):
        def odd(n):
            t = torch.empty(int(n) + 512, dtype=torch.uint8, device="cuda")
            return t, t.data_ptr() + 8
        ocn.Model(wl, workspace=odd)
