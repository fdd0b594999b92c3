"""Writes tests/golden/config0_oracle_summary.txt from the CPU oracle alone (never the CUDA path)."""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import tpc_oracle as orc  # noqa: E402
from paper_2106_03636_b200.synth import config0  # noqa: E402

ev = config0()
o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
lines = [
    "# configs[0] (seed 1) through oracle/tpc_oracle.cpp, real_t = float; written by make_config0_summary.py",
    f"n_clusters {ev.n}",
    f"n_start_hits {o['starts'].size}",
    f"n_tracks {o['trk_seed'].size}",
    f"n_assigned {(o['cluster_track'] >= 0).sum()}",
    f"sum_trk_nhits {int(o['trk_nhits'].sum())}",
    f"sha256_cluster_seed {hashlib.sha256(np.where(o['cluster_track'] >= 0, o['trk_seed'][np.maximum(o['cluster_track'], 0)], -1).astype(np.int32).tobytes()).hexdigest()}",
]
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle_summary.txt"), "w") as f:
    f.write("\n".join(lines) + "\n")
print("\n".join(lines))
