"""Where the warps of the tendency kernel spend their cycles (diagnostic build of libocn only).

    OCN_NVCC_FLAGS=-DOCN_K1_TIMELINE python -m paper_2309_06662_b200.build --force
    python -m paper_2309_06662_b200.timeline [--config 4] [--closure ri]

Prints, per warp of the 256-thread CTA, the average SM cycles per iteration of the march (one level) spent in each phase,
from ocn_get_timeline.  BAR.SYNC does not block at issue, so the time a warp waits for the slowest warp of the level is
booked on the phase after the barrier ("prologue+barrier_wait").  Rebuild without the flag afterwards.
"""
import argparse

from . import ocn, workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--closure", default="const", choices=["const", "ri"])
    ap.add_argument("--patch", default="16x4", help="config 6 only: WxH ocean patch of every 32x8 tile")
    a = ap.parse_args()
    if a.config == 6:
        pw, ph = (int(x) for x in a.patch.lower().split("x"))
        wl = W.make(6, w=pw, h=ph)
    else:
        wl = W.make(a.config)
    if a.closure == "ri":
        W.with_ri_closure(wl)
    m = ocn.Model(wl)
    m.time_step(3)
    m.timeline(reset=True)
    m.time_step(2)
    rows = m.timeline(reset=True)
    names = list(rows[0])
    print("config %d (%s), cycles per iteration per warp" % (a.config, wl["name"]))
    print("warp  " + "  ".join("%22s" % n for n in names) + "   busy (phase1+faces+partB)   total")
    for w, r in enumerate(rows):
        busy = r["phase1"] + r["faces"] + r["partB"]
        print("%4d  " % w + "  ".join("%22.0f" % r[n] for n in names) + "   %8.0f   %8.0f" % (busy, sum(r.values())))
    mean = {n: sum(r[n] for r in rows) / len(rows) for n in names}
    busy = mean["phase1"] + mean["faces"] + mean["partB"]
    print("mean  " + "  ".join("%22.0f" % mean[n] for n in names) + "   %8.0f   %8.0f" % (busy, sum(mean.values())))
    m.close()


if __name__ == "__main__":
    main()
