"""A small case for `compute-sanitizer --tool racecheck|memcheck|synccheck python tests/sanitizer_case.py` (DESIGN.md
section 9): configs[0] with both exact sweep variants, persistent and per-interval launches, a swap event every sweep."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_1308_5426_b200 import inputs, pt  # noqa: E402

w = inputs.config(0)
for variant in ("direct", "field"):
    g = pt.PT(w.L, w.q, w.sigma, 1, w.n_rep, inputs.betas(w), w.seed, variant=variant)
    g.sweeps(1, 1)
    g.sweeps(6, 1)
    assert (g.energy() == g.energy(recompute=True)).all()
    g.close()
print("sanitizer_case OK")
