"""Tiny runs of every kernel family for compute-sanitizer: `compute-sanitizer --tool memcheck|racecheck
python tests/sanitizer_cases.py`.  Not a pytest module (no test_ prefix): the parity of the same cases is checked by the
-m gpu tests; here only the sanitizer's verdict matters."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2501_05440_b200 import binding, inputs  # noqa: E402


def main():
    cases = [
        ("C1 default", inputs.config1(n_particles=600, n_inactive=1, n_active=1), dict()),
        ("C4small sweeps", inputs.config4(n_particles=600, n_inactive=1, n_active=1, n_asm=1, n_pin=3, n_refl=1), dict(persist_threshold=-1)),
        ("C4small monolithic", inputs.config4(n_particles=400, n_inactive=0, n_active=2, n_asm=1, n_pin=3, n_refl=1), dict(schedule=1)),
        ("C4 two-level", inputs.config4(n_particles=500, n_inactive=1, n_active=1, n_asm=1, n_pin=3, n_refl=3, two_level=True), dict()),
        ("mixed split kernels", inputs.mixed_surfaces(n_particles=500), dict(schedule=2, persist_threshold=-1)),
        ("C3 implicit capture", dict(inputs.config3(n_particles=500, n_inactive=1, n_active=1), implicit_capture=1), dict()),
        ("C5 persistent", inputs.config5(n_particles=150, n_grid=3000), dict(search=1)),
        ("C5 sweeps", inputs.config5(n_particles=100, n_grid=3000), dict(persist_threshold=-1)),
        ("TD comb", inputs.td_infinite(n_particles=400, G=2, geom="pin", census_target=300), dict()),
    ]
    for name, P, kw in cases:
        g = binding.Problem(P, **kw)
        r = g.run()
        print(name, "ok", int(r["counters"][1:10].sum()), "events", flush=True)
        g.close()
    P = inputs.config5(n_particles=100, n_grid=3000)
    g = binding.Problem(P)
    for k in range(len(P["t_edges"]) - 1):
        g.run_cycle(100, k, 1, 1)
    print("C5 by intervals ok", flush=True)
    g.close()


if __name__ == "__main__":
    main()
