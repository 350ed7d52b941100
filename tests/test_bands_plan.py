"""CPU tests of the latitude-band orchestration (paper_2309_06662_b200/bands.py): the exchange plan as index
logic, the sliced workloads, and the protocol itself — parts of a step, which rows travel after which part — on a
stand-in "model" (numpy, a few lines, NOT the method) whose parts have the same reach structure as the real ones, run
(a) as several bands in one process and (b) as one band per rank over gloo, world size 2 and 3.  Equality with the
whole-grid stand-in is exact, as it is on the GPU between band models and the whole-grid model (tests/test_gpu_bands.py)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2309_06662_b200 import bands, workloads as W


# ---------------------------------------------------------------------------- the plan
@pytest.mark.parametrize("ny,nb,h", [(75, 3, 14), (600, 8, 14), (40, 2, 10), (41, 4, 10), (1200, 8, 14), (30, 1, 14)])
def test_plan_fills_every_overlap_row_once_from_its_owner(ny, nb, h):
    own, ext, tr = bands.exchange_plan(ny, nb, h)
    assert own[0][0] == 0 and own[-1][1] == ny and all(own[b][1] == own[b + 1][0] for b in range(nb - 1))
    assert max(o[1] - o[0] for o in own) - min(o[1] - o[0] for o in own) <= 1
    owner = np.empty(ny, int)
    for b, o in enumerate(own):
        owner[o[0]:o[1]] = b
    filled = [np.zeros(e[1] - e[0], int) for e in ext]
    for t in tr:
        assert t.nrows > 0 and 0 <= t.src_row and t.src_row + t.nrows <= ext[t.src][1] - ext[t.src][0]
        assert 0 <= t.dst_row and t.dst_row + t.nrows <= ext[t.dst][1] - ext[t.dst][0]
        gs = ext[t.src][0] + t.src_row                      # same global rows on both sides, owned by the source
        assert gs == ext[t.dst][0] + t.dst_row
        assert (owner[gs:gs + t.nrows] == t.src).all()
        filled[t.dst][t.dst_row:t.dst_row + t.nrows] += 1
    for b in range(nb):
        glob = np.arange(ext[b][0], ext[b][1])
        is_own = (glob >= own[b][0]) & (glob < own[b][1])
        assert (filled[b][is_own] == 0).all() and (filled[b][~is_own] == 1).all()
        assert ext[b][0] == max(own[b][0] - h, 0) and ext[b][1] == min(own[b][1] + h, ny)


def test_plan_rejects_bands_thinner_than_the_overlap():
    with pytest.raises(ValueError, match="fewer than the overlap"):
        bands.exchange_plan(40, 4, 14)
    with pytest.raises(ValueError):
        bands.band_rows(10, 11)


def test_groups_follow_the_parts():
    # 4 launches (fp32, M = 40): K1, 4 launches, end
    assert [bands.group_after_part(p, 6) for p in range(6)] == [bands.FORCING, bands.BAROTROPIC_0 + 1, bands.BAROTROPIC_0,
                                                                 bands.BAROTROPIC_0 + 1, None, bands.STATE]
    assert [bands.group_after_part(p, 3) for p in range(3)] == [bands.FORCING, None, bands.STATE]


def test_band_workload_slices_rows_and_keeps_whole_grid_row_numbers():
    wl = W.make(3, nx=48, ny=40, nz=6)
    b = bands.band_workload(wl, (12, 31))
    assert b["grid"]["ny"] == 19 and b["grid"]["j_offset"] == 12 and b["grid"]["ny_global"] == 40
    assert b["grid"]["y0"] == wl["grid"]["y0"] and b["grid"]["periodic_y"] == 0
    assert np.array_equal(b["depth"], wl["depth"][12:31])
    for k, v in wl["fields"].items():
        assert np.array_equal(b["fields"][k], v[..., 12:31, :])
    assert wl["grid"]["ny"] == 40 and "j_offset" not in wl["grid"]          # the source is not modified
    bb = bands.band_workload(b, (3, 10))                                       # a band of a band
    assert bb["grid"]["j_offset"] == 15 and bb["grid"]["ny_global"] == 40
    with pytest.raises(ValueError, match="bounded in y"):
        bands.band_workload(W.make(0), (0, 16))


# ---------------------------------------------------------------------------- the protocol on a stand-in model
SUB, REACH0 = 5, 3            # rows one "launch" and the "tendency" part reach; every exchange resets the overlap rows, so the
H = max(SUB, REACH0)          # reaches do not add up: the overlap is the largest reach of one part
NLAUNCH = 3


class StandIn:
    """A 2-field toy with the reach structure of a step: part 0 builds b from a with a (2 REACH0 + 1)-row stencil, each of
    NLAUNCH middle parts smooths b SUB times by one row each way (walls at the ends of ITS rows), the last part adds b to a.
    pack / unpack move rows of a (STATE) or b (any other group) through a CPU uint8 tensor."""

    def __init__(self, wl, stream=None):
        self.a = np.array(wl["fields"]["eta"], dtype=np.float64)
        self.b = np.zeros_like(self.a)
        self.nx = self.a.shape[1]

    def step_parts(self):
        return NLAUNCH + 2

    def step_part(self, part):
        if part == 0:
            p = np.pad(self.a, ((REACH0, REACH0), (0, 0)))
            self.b = sum((q + 1.0) * p[q:q + self.a.shape[0]] for q in range(2 * REACH0 + 1)) / 16.0
        elif part <= NLAUNCH:
            for _ in range(SUB):
                p = np.pad(self.b, ((1, 1), (0, 0)))
                self.b = 0.25 * p[:-2] + 0.5 * p[1:-1] + 0.25 * p[2:] + 0.01 * np.roll(self.b, 1, axis=1)
        else:
            self.a = self.a + 0.125 * self.b

    def _arr(self, group):
        return self.a if group == bands.STATE else self.b

    def rows_bytes(self, group, nrows):
        return nrows * self.nx * 8

    def pack_rows(self, group, j, n, buf):
        buf.numpy().view(np.float64)[:] = self._arr(group)[j:j + n].ravel()

    def unpack_rows(self, group, j, n, buf):
        self._arr(group)[j:j + n] = buf.numpy().view(np.float64).reshape(n, self.nx)

    def get_fields(self, names):
        return {"eta": self.a.copy()}

    def synchronize(self):
        pass

    def close(self):
        pass


def _toy_workload(ny=67, nx=9, seed=5):
    rng = np.random.default_rng(seed)
    return dict(name="toy", grid=dict(ny=ny, nx=nx, periodic_y=0), depth=np.ones((ny, nx)),
                params=dict(precision=64, substeps=SUB * NLAUNCH), fields=dict(eta=rng.standard_normal((ny, nx))))


def _alloc(nbytes):
    t = torch.empty(int(nbytes), dtype=torch.uint8)
    return t, t


def _whole(wl, steps):
    m = StandIn(wl)
    for _ in range(steps):
        for p in range(m.step_parts()):
            m.step_part(p)
    return m.a


@pytest.mark.parametrize("nb", [1, 2, 3, 5])
def test_bands_in_one_process_reproduce_the_whole_grid_exactly(nb):
    wl = _toy_workload()
    B = bands.Bands(wl, nb, h=H, model_factory=lambda w, s: StandIn(w), alloc=_alloc)
    B.time_step(4)
    assert np.array_equal(B.get_fields(("eta",))["eta"], _whole(wl, 4))


def test_an_overlap_one_row_short_is_caught():
    wl = _toy_workload()
    B = bands.Bands(wl, 3, h=H - 1, model_factory=lambda w, s: StandIn(w), alloc=_alloc)
    B.time_step(4)
    assert not np.array_equal(B.get_fields(("eta",))["eta"], _whole(wl, 4))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = _toy_workload()
        D = bands.DistBand(wl, dist, h=H, model_factory=lambda w, s: StandIn(w), alloc=_alloc)
        D.time_step(4)
        out.put((rank, D.own[rank], D.own_fields(("eta",))["eta"]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_one_band_per_rank_over_gloo_reproduces_the_whole_grid_exactly(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=180) for _ in ps), key=lambda r: r[0])
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = _whole(_toy_workload(), 4)
    for rank, own, a in res:
        assert np.array_equal(a, ref[own[0]:own[1]]), rank
    assert res[0][1][0] == 0 and res[-1][1][1] == ref.shape[0]
