"""Operation counts of O4 per tracklet hit, for the measurement's algorithmic operation count.

TEST INFRASTRUCTURE: calls only `oracle/` and the seeded input generator.  Run as

    python oracle/count_o4_ops.py [config] [sector ...]

It prints, per sampled sector of the synthetic event, how often the oracle's O4 ran Propagate, Update and Search, how many
clusters its Searches found inside their roads, and the four counts per hit of the accepted tracklets (the unit `bench.py`
multiplies by: `n_tracklet_hits` of the run status).  The per-hit figures quoted in DESIGN.md section 8 and used by
`bench.py` (`O4_OPS_PER_HIT`) are the config-4 output of this script.
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from oracle import tpc_oracle as orc                      # noqa: E402
from paper_1910_12214_b200 import datagen                 # noqa: E402


def main(argv):
    config = int(argv[1]) if len(argv) > 1 else 4
    sectors = [int(a) for a in argv[2:]] or [0, 7, 20]
    ev = datagen.make_event(config)
    R = ev.n_rows
    for sct in sectors:
        if ev.n_sectors == 1:
            s = ev
        else:
            lo, hi = int(ev.row_offset[sct * R]), int(ev.row_offset[(sct + 1) * R])
            o = (ev.row_offset[sct * R:(sct + 1) * R + 1].astype(np.int64) - lo).astype(np.uint32)
            s = datagen.event_from_arrays(o, ev.y[lo:hi], ev.z[lo:hi], 1, R, row_x=ev.row_x, z_min=ev.z_min,
                                          z_max=ev.z_max, bz_tesla=ev.bz_tesla)
        r = orc.run(s)
        H = int(r.tl_nhits[r.tl_status == 2].sum())
        print(f"config {config} sector {sct}: clusters {s.n_clusters}  Propagate/Update/Search/in-road {r.o4_ops.tolist()}"
              f"  accepted tracklet hits {H}  per hit {np.round(r.o4_ops / max(H, 1), 4).tolist()}")


if __name__ == "__main__":
    main(sys.argv)
