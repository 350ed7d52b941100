"""GPU tests of the latitude-band form of the path (include/ocn.h "Latitude bands"): a
grid stepped as 2, 3 or 4 band models that exchange overlap rows after each part of a step gives, on every band's own
rows, the SAME BITS as the whole-grid model (which the other GPU tests hold against the oracle) — fp64 and fp32, with the
closure, bottom drag and the biharmonic terms, and the fp64 bands are therefore bit-identical to the oracle as well.
One GPU, one stream: this is the decomposition made correct by construction; the same plan over torch.distributed is
covered on CPU (tests/test_bands_plan.py)."""
import ctypes as C

import numpy as np
import pytest

import oracle
from paper_2309_06662_b200 import bands
from paper_2309_06662_b200 import build as ocn_build
from paper_2309_06662_b200 import ocn
from paper_2309_06662_b200 import workloads as W

pytestmark = pytest.mark.gpu
FIELDS = ("u", "v", "w", "eta", "T", "S")


@pytest.fixture(scope="module", autouse=True)
def _built():
    ocn_build.build()


def _stirred(wl, seed=33):
    rng = np.random.default_rng(seed)
    f, prec = wl["fields"], wl["params"]["precision"]
    f["u"] = W._round_to(prec, 0.3 * rng.standard_normal(f["u"].shape))
    f["v"] = W._round_to(prec, 0.3 * rng.standard_normal(f["v"].shape))
    f["T"] = W._round_to(prec, f["T"] + 0.5 * rng.standard_normal(f["T"].shape))
    f["eta"] = W._round_to(prec, 0.2 * rng.standard_normal(f["eta"].shape))
    return wl


def _workload(prec, kind=""):
    wl = _stirred(W.config2(nx=180, ny=75, nz=25, steps=6, precision=prec))
    if "r" in kind:
        W.with_ri_closure(wl)
    if "d" in kind:
        wl["params"].update(drag_r=2e-4, drag_cd=2e-3)
    if "b" in kind:
        wl["params"].update(nu4_h=1e9, kappa4_h=5e8)
    if "z" in kind:
        W.with_weno_z(wl)
    return wl


def test_the_parts_of_a_step_are_the_step():
    for prec in (32, 64):
        wl = _workload(prec, "r")
        a, b = ocn.Model(wl), ocn.Model(wl)
        a.time_step(5)
        n = b.step_parts()
        assert n == b.info()["launches_per_step"] - 1              # K1, the launches of the sub-cycle, [finish + K3]
        for _ in range(5):
            for p in range(n):
                b.step_part(p)
        fa, fb = a.get_fields(), b.get_fields()
        for k in FIELDS:
            assert np.array_equal(fa[k], fb[k]), (prec, k)
        a.close(); b.close()


def test_parts_run_in_order_and_block_whole_steps():
    m = ocn.Model(_workload(32))
    with pytest.raises(RuntimeError, match="parts of a step run in order"):
        m.step_part(1)
    m.step_part(0)
    with pytest.raises(RuntimeError, match="split step is in progress"):
        m.time_step(1)
    with pytest.raises(RuntimeError, match="parts of a step run in order"):
        m.step_part(0)
    with pytest.raises(RuntimeError, match="no such part"):
        m.step_part(m.step_parts())
    for p in range(1, m.step_parts()):
        m.step_part(p)
    m.time_step(1)                                                 # the step is complete: whole steps are allowed again
    m.close()


def test_rows_round_trip_and_are_checked():
    import torch
    wl = _workload(64)
    a, b = ocn.Model(wl), ocn.Model(wl)
    a.time_step(3); b.time_step(1)                                 # different states
    for group in (ocn.ROWS_STATE, ocn.ROWS_STATE_2D, ocn.ROWS_FORCING, ocn.ROWS_BAROTROPIC_0, ocn.ROWS_BAROTROPIC_1):
        nb = a.rows_bytes(group, a.ny)
        buf = torch.empty(nb, dtype=torch.uint8, device="cuda")
        a.synchronize(); b.synchronize()
        a.pack_rows(group, 0, a.ny, buf.data_ptr())
        a.synchronize()
        b.unpack_rows(group, 0, b.ny, buf.data_ptr())
        b.synchronize()
    fa, fb = a.get_fields(("u", "v", "T", "S", "eta")), b.get_fields(("u", "v", "T", "S", "eta"))
    for k in fa:
        assert np.array_equal(fa[k], fb[k]), k                     # every row of the state travelled
    sx = (a.nx + 8 + 31) // 32 * 32
    assert a.rows_bytes(ocn.ROWS_FORCING, 7) == 2 * 7 * sx * 8
    assert a.rows_bytes(ocn.ROWS_STATE, 2) == 2 * sx * (25 * (16 + 16 + 8) + 3 * 8)
    assert a.rows_bytes(ocn.ROWS_STATE_2D, 2) == 2 * sx * 3 * 8
    with pytest.raises(RuntimeError, match="rows outside the grid"):
        a.pack_rows(ocn.ROWS_STATE, a.ny - 2, 3, buf.data_ptr())
    with pytest.raises(RuntimeError, match="unknown row group"):
        a.rows_bytes(9, 1)
    assert ocn.band_overlap(32, 40) == 11 and ocn.band_overlap(64, 40) == 7 and ocn.band_overlap(64, 2) == 4
    a.close(); b.close()


def test_band_masks_are_the_whole_grids_away_from_its_walls():
    wl = _workload(64)
    g = ocn.Grid(wl["grid"], wl["z_faces"], wl["depth"])
    bw = bands.band_workload(wl, (20, 51))
    gb = ocn.Grid(bw["grid"], bw["z_faces"], bw["depth"])
    mw, mb = g.masks(), gb.masks()
    inner = slice(3, 31 - 3)                                       # away from the band's artificial walls
    for k in mw:
        assert np.array_equal(mw[k][:, 20:51][:, inner], mb[k][:, inner]), k
    bad = dict(bw["grid"], ny_global=40)
    with pytest.raises(RuntimeError, match="band must lie inside"):
        ocn.Grid(bad, bw["z_faces"], bw["depth"])


@pytest.mark.parametrize("prec,kind,nb", [(64, "", 2), (64, "r", 3), (64, "db", 3), (32, "", 2), (32, "r", 3), (32, "dbz", 4), (32, "", 1)])
def test_bands_are_bit_identical_to_the_whole_grid(prec, kind, nb):
    wl = _workload(prec, kind)
    whole = ocn.Model(wl)
    B = bands.Bands(wl, nb)
    assert B.h == ocn.band_overlap(prec, wl["params"]["substeps"])
    whole.time_step(6); B.time_step(6)
    fw, fb = whole.get_fields(), B.get_fields()
    for k in FIELDS:
        assert fb[k].shape == fw[k].shape
        assert np.array_equal(fw[k], fb[k]), (prec, kind, nb, k, float(np.abs(fw[k].astype(np.float64) - fb[k]).max()))
    assert float(np.abs(fw["u"]).max()) > 0.05 and np.isfinite(fw["T"]).all()
    whole.close(); B.close()


def test_fp64_bands_are_bit_identical_to_the_oracle():
    wl = _workload(64, "r")
    ref = oracle.RefModel(wl)
    B = bands.Bands(wl, 3)
    ref.step(6); B.time_step(6)
    a, b = B.get_fields(), ref.get_fields()
    for k in FIELDS:
        assert np.array_equal(a[k], b[k]), k
    B.close()


def test_exchanged_bytes_per_step_are_what_the_design_says():
    wl = _workload(32)
    B = bands.Bands(wl, 3)
    m = B.models[0]
    per = {g: m.rows_bytes(g, B.h) for g in (ocn.ROWS_STATE, ocn.ROWS_FORCING, ocn.ROWS_BAROTROPIC_0)}
    groups = [bands.group_after_part(p, B.parts) for p in range(B.parts)]
    total = sum(per[min(g, ocn.ROWS_BAROTROPIC_0)] for g in groups if g is not None)
    sx = (m.nx + 8 + 31) // 32 * 32
    nz = m.nz
    # per cut and direction: h rows of (u,v), (T,S) pairs + p (fp64) + eta, U, V once; G^U, G^V once; eta, U, V after every launch but the last
    launches = B.parts - 2
    assert total == B.h * sx * (nz * (8 + 8 + 8) + 3 * 4 + 2 * 4 + (launches - 1) * 3 * 4)
    B.close()


# ---- one band per PROCESS: two ranks share this one GPU, the packed rows travel through pinned host memory over gloo (NCCL
# cannot put two ranks on one device).  No kernel of one rank waits for a kernel of the other: the ranks meet on the host.
def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_worker(rank, world, port, prec, kind, steps, out):
    import os
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            D = bands.DistBand(_workload(prec, kind), dist, device=0, stream=s.cuda_stream, host_staging=True)
            D.time_step(steps)
            f = D.own_fields(FIELDS)
        out.put((rank, D.own[rank], {k: np.array(v) for k, v in f.items()}))
        dist.barrier()
        D.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("prec,kind,world", [(32, "r", 2), (64, "", 3)])
def test_one_band_per_process_is_bit_identical_to_the_whole_grid(prec, kind, world):
    import torch.multiprocessing as mp
    steps = 4
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_rank_worker, args=(r, world, port, prec, kind, steps, q)) for r in range(world)]
    for p in ps:
        p.start()
    whole = ocn.Model(_workload(prec, kind))
    whole.time_step(steps)
    fw = whole.get_fields()
    whole.close()
    res = sorted((q.get(timeout=600) for _ in ps), key=lambda r: r[0])
    for p in ps:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert res[0][1][0] == 0 and res[-1][1][1] == fw["eta"].shape[0]
    for rank, own, f in res:
        for k in FIELDS:
            assert np.array_equal(f[k], fw[k][..., own[0]:own[1], :]), (rank, k)


def test_bench_bands_line():
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--bands", "3", "--config", "3", "--steps", "2", "--warmup", "3"],
                       capture_output=True, text=True, timeout=900, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    b = d["bands"]
    assert b["n"] == 3 and b["overlap_rows"] == 11 and sum(b["own_rows"]) == 600 and b["exchanges_per_step"] == b["parts_per_step"] - 1
    assert b["ms_per_step_per_band"] > 0 and 1.0 < b["projected_speedup_on_n_gpus"] < 3.0


# ---- fused puts: the last part of a step stores the overlap rows of the neighbours itself (no exchange of the new state) ----
@pytest.mark.parametrize("prec,kind,nb", [(64, "r", 3), (64, "db", 2), (32, "", 2), (32, "r", 4), (32, "dbz", 3)])
def test_bands_with_fused_puts_are_bit_identical_to_the_whole_grid(prec, kind, nb):
    wl = _workload(prec, kind)
    whole = ocn.Model(wl)
    B = bands.Bands(wl, nb, fused_put=True)
    whole.time_step(6); B.time_step(6)
    fw, fb = whole.get_fields(), B.get_fields()
    for k in FIELDS:
        assert np.array_equal(fw[k], fb[k]), (prec, kind, nb, k)
    whole.close(); B.close()


def test_peer_attach_is_checked():
    a, b = ocn.Model(_workload(32)), ocn.Model(_workload(64))
    with pytest.raises(RuntimeError, match="same nx, nz and precision"):
        a.peer_attach(0, b.peer_export(), 0, 0, 4, True)
    c = ocn.Model(_workload(32))
    with pytest.raises(RuntimeError, match="rows outside a grid"):
        a.peer_attach(1, c.peer_export(), a.ny - 2, 0, 4, True)
    with pytest.raises(RuntimeError, match="side must be"):
        a.peer_attach(2, c.peer_export(), 0, 0, 4, True)
    for m in (a, b, c):
        m.close()


def _rank_worker_put(rank, world, port, prec, kind, steps, out):
    import os
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        D = bands.DistBand(_workload(prec, kind), dist, device=0, host_staging=True, fused_put=True)   # on a stream of its own
        D.time_step(steps)
        f = D.own_fields(FIELDS)
        out.put((rank, D.own[rank], {k: np.array(v) for k, v in f.items()}))
        dist.barrier()
        D.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("prec,kind,world", [(32, "r", 2), (64, "", 3)])
def test_fused_puts_across_processes_through_cuda_ipc(prec, kind, world):
    """One band per process, all on this one GPU: the new state reaches the neighbour through CUDA IPC mappings written by the
    producing kernels; the small 2-D groups and the per-step tokens travel over gloo."""
    import torch.multiprocessing as mp
    steps = 4
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_rank_worker_put, args=(r, world, port, prec, kind, steps, q)) for r in range(world)]
    for p in ps:
        p.start()
    whole = ocn.Model(_workload(prec, kind))
    whole.time_step(steps)
    fw = whole.get_fields()
    whole.close()
    res = sorted((q.get(timeout=600) for _ in ps), key=lambda r: r[0])
    for p in ps:
        p.join(timeout=120)
        assert p.exitcode == 0
    for rank, own, f in res:
        for k in FIELDS:
            assert np.array_equal(f[k], fw[k][..., own[0]:own[1], :]), (rank, k)


def test_forcing_that_changes_between_steps_reaches_every_band():
    wl = _workload(32, "r")
    whole = ocn.Model(wl)
    B = bands.Bands(wl, 3)
    rng = np.random.default_rng(8)
    for n in range(3):
        tx = (0.1 * rng.standard_normal(wl["fields"]["tau_x"].shape)).astype(np.float32)
        qT = (1e-5 * rng.standard_normal(tx.shape)).astype(np.float32)
        whole.set_fields(tau_x=tx, flux_T=qT)
        B.set_forcing(tau_x=tx, flux_T=qT)
        whole.time_step(2); B.time_step(2)
    fw, fb = whole.get_fields(), B.get_fields()
    for k in FIELDS:
        assert np.array_equal(fw[k], fb[k]), k
    with pytest.raises(ValueError, match="set_forcing takes"):
        B.set_forcing(u=wl["fields"]["u"])
    whole.close(); B.close()


def test_the_overlap_is_the_smallest_that_keeps_the_bits_in_fp64():
    """ocn_band_overlap is the reach of one part + 1: with one row less the error of the band's artificial wall arrives on own
    rows within a launch of the sub-cycle (1e-16 relative after six sub-steps, but not the same bits).  (In fp32 the same
    intrusion falls below the rounding of the fields for a few rows more; the overlap there is the bound, not the observation.)"""
    wl = _workload(64, "")
    whole = ocn.Model(wl)
    whole.time_step(6)
    fw = whole.get_fields()
    whole.close()
    h = ocn.band_overlap(64, wl["params"]["substeps"])
    B = bands.Bands(wl, 3, h=h - 1)
    B.time_step(6)
    fb = B.get_fields()
    B.close()
    assert not np.array_equal(fw["eta"], fb["eta"])
    assert np.abs(fw["eta"] - fb["eta"]).max() < 1e-12


@pytest.mark.parametrize("nb,fused", [(2, False), (8, True)])
def test_bands_at_the_full_size_of_config_4_are_bit_identical(nb, fused):
    """The grid bench.py times (2880 x 1200 x 100, fp32, M = 40), cut into 2 bands with packed-row exchange and into 8 bands with
    fused puts: the same bits as one model after an Euler step and three quasi-AB2 steps."""
    wl = W.make(4)
    names = ("u", "v", "T", "eta")
    whole = ocn.Model(wl)
    whole.time_step(4)
    fw = whole.get_fields(names)
    whole.close()
    B = bands.Bands(wl, nb, fused_put=fused)
    B.time_step(4)
    fb = B.get_fields(names)
    B.close()
    for k in names:
        assert np.array_equal(fw[k], fb[k]), (nb, fused, k)
    assert float(np.abs(fw["u"]).max()) > 1e-3
