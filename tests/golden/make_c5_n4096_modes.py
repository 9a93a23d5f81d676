"""Writes tests/golden/c5_n4096_oracle_modes.txt: the mode set the fp64 oracle returns on the reduced end-to-end
run SURVEY.md section 8(d) prescribes for C5 ("same d, K; N = 4096, 10 cycles"), noise-free (R-14).

Calls only oracle/ (and the seeded input generator); nothing here comes from the CUDA path.  Takes ~1 h on 8 cores:
    python tests/golden/make_c5_n4096_modes.py [threads]
The run parameters are those of tests/test_gpu_end_to_end.py::C5_E2E (kept in one place: E2E_OVERRIDES below).
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)

import oracle as O                                   # noqa: E402
from paper_2606_26164_b200 import inputs             # noqa: E402

# noise-free thresholds: eps_grad bounds the position error of a frozen sample by eps_grad / curvature (curvature
# >= 1 / 0.5 at C5), so 5e-4 keeps it under 1e-3 L2; log_delta = -30 keeps every component peak in M* (Eq. 1)
E2E_N, E2E_CYCLES = 4096, 10
E2E_OVERRIDES = dict(eps_grad=5e-4, eps_dup=1e-2, log_delta=-30.0, n_conv=60)
OUT = os.path.join(HERE, "c5_n4096_oracle_modes.txt")


def main():
    threads = int(sys.argv[1]) if len(sys.argv) > 1 else len(os.sched_getaffinity(0))
    wl = inputs.config(5, N=E2E_N, n_osc=E2E_CYCLES, noise=0.0, **E2E_OVERRIDES)
    o = O.Oracle(wl, threads=threads)
    per_cycle = []
    t0 = time.time()
    for k in range(E2E_CYCLES):
        st = o.step()
        per_cycle.append((st.cycle, st.n_stuck, st.k_lost, st.n_active, st.reseed_strategy))
        print(per_cycle[-1], f"{time.time() - t0:.0f} s", flush=True)
    x, f, idx = o.modes()
    with open(OUT, "w") as fh:
        fh.write("# fp64 oracle, C5 noise-free, N = 4096, 10 cycles; written by tests/golden/make_c5_n4096_modes.py\n")
        fh.write("# per cycle (cycle, n_stuck, k_lost, n_active, strategy): " + " ".join(map(str, per_cycle)) + "\n")
        fh.write(f"# {len(f)} modes; columns: sample index, f, x[0..63]\n")
        for q in range(len(f)):
            fh.write(" ".join([str(int(idx[q])), repr(float(f[q]))] + [repr(float(v)) for v in x[q]]) + "\n")
    print("wrote", OUT, len(f), "modes")


if __name__ == "__main__":
    main()
