"""Latitude bands: the sharded form of the path.

The whole grid is cut into bands of rows; every band is an ordinary model (`ocn.Model`) on its own rows plus `h` overlap
rows on each inner side, built with `ocn_grid_desc.j_offset / ny_global` so that its metrics are the whole grid's.  A
step runs in parts (`ocn_step_part`); after each part the overlap rows are overwritten with the neighbour's own rows of
the arrays that part made stale (`ocn_pack_rows` / `ocn_unpack_rows`), so that every band's own rows stay bit-identical
to the whole-grid model.  This is the paper's scheme (the barotropic mode is stepped with a wide halo so
that neighbours talk once per group of sub-steps; the 3-D halos once per step) with the overlap rows also
standing in for the paper's halo regions.

This module is orchestration only: which rows go where and in what order.  All arithmetic is in the kernels; the bytes
move by device-to-device copies (same process) or by torch.distributed point-to-point calls (one band per rank: NCCL on
GPUs, gloo in the CPU test of the plan).  It holds none of the method's arithmetic and never touches the oracle.

    Bands(workload, nbands)         all bands in this process, on one stream of one GPU (tests, single-GPU runs)
    DistBand(workload, dist)        this rank's band; neighbours are ranks +-1
"""
from __future__ import annotations

import numpy as np

from . import ocn

STATE, FORCING, BAROTROPIC_0, STATE_2D = ocn.ROWS_STATE, ocn.ROWS_FORCING, ocn.ROWS_BAROTROPIC_0, ocn.ROWS_STATE_2D


# ------------------------------------------------------------------------------------------------
# the plan: pure index logic (covered on CPU by tests/test_bands_plan.py)
# ------------------------------------------------------------------------------------------------
def band_rows(ny, nbands):
    """Own rows [lo, hi) of each band: as even as integers allow, the taller bands first."""
    if nbands < 1 or nbands > ny:
        raise ValueError("nbands must be in 1 .. ny")
    q, r = divmod(int(ny), int(nbands))
    out, lo = [], 0
    for b in range(nbands):
        hi = lo + q + (1 if b < r else 0)
        out.append((lo, hi))
        lo = hi
    return out


def band_extent(own, ny, h):
    """Rows [lo, hi) the band's model covers: its own rows + h overlap rows towards each neighbour, clipped to the grid."""
    return max(own[0] - h, 0), min(own[1] + h, ny)


def group_after_part(part, parts):
    """Row group to exchange after part `part` of a step of `parts` parts (include/ocn.h, "Latitude bands"); None = nothing."""
    if part == 0:
        return FORCING
    if part == parts - 1:
        return STATE
    if part == parts - 2:
        return None                       # the last launch of the sub-cycle: only its filtered sums are used, on own rows
    return BAROTROPIC_0 + (part & 1)      # launch q = part - 1 wrote buffer (q + 1) & 1 = part & 1


class Transfer:
    """`nrows` rows starting at local row `src_row` of band `src` -> local row `dst_row` of band `dst`."""
    __slots__ = ("src", "src_row", "dst", "dst_row", "nrows")

    def __init__(self, src, src_row, dst, dst_row, nrows):
        self.src, self.src_row, self.dst, self.dst_row, self.nrows = src, src_row, dst, dst_row, nrows

    def __repr__(self):
        return "Transfer(%d:%d -> %d:%d, %d rows)" % (self.src, self.src_row, self.dst, self.dst_row, self.nrows)


def exchange_plan(ny, nbands, h):
    """(own, extent, transfers): every overlap row of every band is filled from the band that owns it."""
    own = band_rows(ny, nbands)
    ext = [band_extent(o, ny, h) for o in own]
    for b in range(nbands):
        inner = (b > 0) + (b < nbands - 1)
        if inner and own[b][1] - own[b][0] < h:
            raise ValueError("band %d owns %d rows, fewer than the overlap of %d rows its neighbour needs" % (b, own[b][1] - own[b][0], h))
    tr = []
    for b in range(nbands - 1):
        n, s = b + 1, b                                    # north and south band of the cut at row own[b][1]
        cut = own[b][1]
        up = ext[s][1] - cut                               # overlap rows of the south band, owned by the north band
        tr.append(Transfer(n, cut - ext[n][0], s, cut - ext[s][0], up))
        dn = cut - ext[n][0]                               # overlap rows of the north band, owned by the south band
        tr.append(Transfer(s, ext[n][0] - ext[s][0], n, 0, dn))
    return own, ext, tr


def band_workload(wl, ext, name=None):
    """The workload restricted to rows ext = [lo, hi) of the whole grid (bounded in y; metrics by whole-grid row numbers)."""
    g = dict(wl["grid"])
    if g.get("periodic_y"):
        raise ValueError("bands cut a grid that is bounded in y")
    lo, hi = ext
    ny = int(g["ny"])
    g.update(ny=hi - lo, j_offset=int(g.get("j_offset", 0)) + lo, ny_global=int(g.get("ny_global", 0)) or ny)
    out = dict(wl)
    out["grid"] = g
    out["name"] = name or "%s[rows %d:%d]" % (wl.get("name", "workload"), lo, hi)
    out["depth"] = np.ascontiguousarray(wl["depth"][lo:hi])
    out["fields"] = {k: np.ascontiguousarray(v[..., lo:hi, :]) for k, v in wl.get("fields", {}).items() if v is not None}
    return out


FORCING_FIELDS = ("tau_x", "tau_y", "flux_T", "flux_S", "restore_T", "restore_S")


def _forcing_only(fields):
    bad = [k for k in fields if k not in FORCING_FIELDS]
    if bad:
        raise ValueError("set_forcing takes %s, not %s" % (", ".join(FORCING_FIELDS), ", ".join(bad)))


def overlap_rows(wl):
    return ocn.band_overlap(wl["params"]["precision"], wl["params"]["substeps"])


# ------------------------------------------------------------------------------------------------
# all bands in one process, one stream (one GPU)
# ------------------------------------------------------------------------------------------------
class Bands:
    """The whole grid as `nbands` band models on ONE stream of one device; results on own rows are those of one model.

    model_factory(workload, stream) builds a band (default: ocn.Model on `device` with that stream); alloc(nbytes) returns
    (handle, device pointer) of a transit buffer (default: a torch uint8 tensor on `device`)."""

    def __init__(self, wl, nbands, device=0, h=None, model_factory=None, alloc=None, stream=None, fused_put=False):
        self.ny = int(wl["grid"]["ny"])
        self.h = overlap_rows(wl) if h is None else int(h)
        self.own, self.ext, self.transfers = exchange_plan(self.ny, nbands, self.h)
        if model_factory is None:
            import torch
            self._stream = torch.cuda.Stream(device=device) if stream is None else stream
            handle = self._stream.cuda_stream
            model_factory = lambda w, s: ocn.Model(w, device=device, stream=s)
            if alloc is None:
                def alloc(nbytes):
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda:%d" % device)
                    return t, t.data_ptr()
        else:
            handle = stream
        self.models = [model_factory(band_workload(wl, e), handle) for e in self.ext]
        self.parts = self.models[0].step_parts()
        self._alloc = alloc
        self._buf = {}
        # fused puts (include/ocn.h): the last part of a step stores the 3-D rows a neighbour overlaps into the neighbour's arrays
        self.fused_put = bool(fused_put) and len(self.models) > 1
        if self.fused_put:
            peers = [m.peer_export() for m in self.models]
            for t in self.transfers:
                self.models[t.src].peer_attach(1 if t.dst > t.src else 0, peers[t.dst], t.src_row, t.dst_row, t.nrows, True)

    def _buffer(self, nbytes):
        if nbytes not in self._buf:
            self._buf[nbytes] = self._alloc(nbytes)
        return self._buf[nbytes][1]

    def exchange(self, group):
        for t in self.transfers:
            if t.nrows == 0:
                continue
            src, dst = self.models[t.src], self.models[t.dst]
            ptr = self._buffer(src.rows_bytes(group, t.nrows))
            src.pack_rows(group, t.src_row, t.nrows, ptr)          # same stream: the unpack follows the pack
            dst.unpack_rows(group, t.dst_row, t.nrows, ptr)

    def time_step(self, n=1):
        for _ in range(int(n)):
            for part in range(self.parts):
                for m in self.models:
                    m.step_part(part)
                g = group_after_part(part, self.parts)
                if g is not None and len(self.models) > 1:
                    self.exchange(STATE_2D if (g == STATE and self.fused_put) else g)

    def set_forcing(self, **fields):
        """Whole-grid forcing fields (tau_x, tau_y, flux_T, flux_S, restore_T, restore_S; host arrays of ny x nx) to every band:
        each gets the rows it covers.  State fields are set through the workload (they restart the time stepping)."""
        _forcing_only(fields)
        for m, e in zip(self.models, self.ext):
            m.set_fields(**{k: np.ascontiguousarray(v[e[0]:e[1]]) for k, v in fields.items()})

    def synchronize(self):
        for m in self.models:
            m.synchronize()

    def get_fields(self, names=("u", "v", "T", "S", "w", "eta")):
        """Own rows of every band, stitched to whole-grid arrays."""
        parts = []
        for m, o, e in zip(self.models, self.own, self.ext):
            f = m.get_fields(names)
            parts.append({k: v[..., o[0] - e[0]:o[1] - e[0], :] for k, v in f.items()})
        return {k: np.concatenate([p[k] for p in parts], axis=-2) for k in names}

    def close(self):
        for m in self.models:
            m.close()
        self.models = []


# ------------------------------------------------------------------------------------------------
# one band per rank (torch.distributed)
# ------------------------------------------------------------------------------------------------
class DistBand:
    """This rank's band of the whole grid; the neighbours are ranks rank - 1 (south) and rank + 1 (north).

    The band's model and torch.distributed's point-to-point calls work on ONE stream, so that the packs, the sends / receives and
    the unpacks are ordered by torch's stream semantics with no host synchronisation: by default a torch stream this object
    creates and makes current around every exchange (torch's legacy default stream has handle 0, which the library would take
    for "give me a private stream"); with `stream` = the handle of a stream of the caller's, that stream must be torch's current
    stream whenever time_step is called.  model_factory / alloc as in Bands; alloc returns (tensor, pointer) and the TENSOR is what is sent.
    host_staging=True: the packed rows travel through pinned host tensors (device -> host, send / recv, host -> device) for
    process groups that cannot send device memory (gloo: the 2-process test on one GPU); the default sends device tensors."""

    def __init__(self, wl, dist, device=0, h=None, model_factory=None, alloc=None, stream=None, host_staging=False,
                 fused_put=False):
        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.ny = int(wl["grid"]["ny"])
        self.h = overlap_rows(wl) if h is None else int(h)
        self.own, self.ext, self.transfers = exchange_plan(self.ny, self.world, self.h)
        if model_factory is None:
            import torch
            self._tstream = torch.cuda.Stream(device=device) if stream is None else None
            handle = self._tstream.cuda_stream if stream is None else stream
            model_factory = lambda w, s: ocn.Model(w, device=device, stream=s)
            if alloc is None:
                def alloc(nbytes):
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda:%d" % device)
                    return t, t.data_ptr()
        else:
            self._tstream = None
            handle = stream
        self.model = model_factory(band_workload(wl, self.ext[self.rank]), handle)
        self.parts = self.model.step_parts()
        self._alloc = alloc
        self._buf = {}
        self._host = {}
        self.host_staging = bool(host_staging)
        # fused puts: the neighbours' arrays are reached through CUDA IPC (one process per GPU on one node); of the new state only
        # the 2-D part is exchanged, and its arrival says that the neighbour's puts (enqueued before its pack) are complete
        self.fused_put = bool(fused_put) and self.world > 1
        if self.fused_put:
            peers = [None] * self.world
            dist.all_gather_object(peers, self.model.peer_export())
            for t in self.transfers:
                if t.src == self.rank:
                    self.model.peer_attach(1 if t.dst > t.src else 0, peers[t.dst], t.src_row, t.dst_row, t.nrows, False)

    def _buffer(self, key, nbytes):
        if (key, nbytes) not in self._buf:
            self._buf[(key, nbytes)] = self._alloc(nbytes)
        return self._buf[(key, nbytes)]

    def _host_buffer(self, key, nbytes):
        import torch
        if (key, nbytes) not in self._host:
            self._host[(key, nbytes)] = torch.empty(int(nbytes), dtype=torch.uint8, pin_memory=True)
        return self._host[(key, nbytes)]

    def exchange(self, group):
        """Sends this band's own edge rows to the neighbours and fills its overlap rows from theirs."""
        if self._tstream is not None:
            import torch
            with torch.cuda.stream(self._tstream):
                return self._exchange(group)
        return self._exchange(group)

    def _exchange(self, group):
        dist = self.dist
        ops, recvs = [], []
        for n, t in enumerate(self.transfers):
            if t.nrows == 0:
                continue
            if t.src == self.rank:
                nbytes = self.model.rows_bytes(group, t.nrows)
                buf, ptr = self._buffer(("s", n), nbytes)
                self.model.pack_rows(group, t.src_row, t.nrows, ptr)
                if self.host_staging:                      # torch's current stream is the model's: the copy follows the pack
                    hb = self._host_buffer(("s", n), nbytes)
                    hb.copy_(buf, non_blocking=True)
                    buf = hb
                ops.append(dist.P2POp(dist.isend, buf, t.dst, tag=n))
            elif t.dst == self.rank:
                nbytes = self.model.rows_bytes(group, t.nrows)
                buf, ptr = self._buffer(("r", n), nbytes)
                hb = self._host_buffer(("r", n), nbytes) if self.host_staging else None
                ops.append(dist.P2POp(dist.irecv, hb if hb is not None else buf, t.src, tag=n))
                recvs.append((t, ptr, buf, hb))
        if ops:
            if self.host_staging:
                self.model.synchronize()                   # the host tensors hold the packed rows before they are sent
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for t, ptr, buf, hb in recvs:
            if hb is not None:
                buf.copy_(hb, non_blocking=True)
            self.model.unpack_rows(group, t.dst_row, t.nrows, ptr)

    def time_step(self, n=1):
        for _ in range(int(n)):
            for part in range(self.parts):
                self.model.step_part(part)
                g = group_after_part(part, self.parts)
                if g is not None and self.world > 1:
                    self.exchange(STATE_2D if (g == STATE and self.fused_put) else g)

    def set_forcing(self, **fields):
        """Whole-grid forcing fields (host arrays of ny x nx): this band takes the rows it covers."""
        _forcing_only(fields)
        e = self.ext[self.rank]
        self.model.set_fields(**{k: np.ascontiguousarray(v[e[0]:e[1]]) for k, v in fields.items()})

    def own_fields(self, names=("u", "v", "T", "S", "w", "eta")):
        """This band's own rows (global rows self.own[rank])."""
        o, e = self.own[self.rank], self.ext[self.rank]
        return {k: v[..., o[0] - e[0]:o[1] - e[0], :] for k, v in self.model.get_fields(names).items()}

    def close(self):
        self.model.close()
