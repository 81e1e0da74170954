"""Full-size, full-length parity run (minutes of CPU time, so not part of the pytest suite):

    python -m tests.full_length_parity config3 config4 sweep_50M

Runs BASELINE.json's config at its full size for its full step count on the GPU (bench.py's
launch configuration) and on the CPU oracle, and prints the largest deviations in the terms of
the parity bar of tests/test_gpu_parity.py (1e-10 relative/absolute on h, hu, hv; 1e-12 relative
on t and dt; identical dry mask).  Exit code 1 if the bar is not met.
"""
import sys
import time

import numpy as np

from oracle.swe_oracle import OracleSolver
from paper_2010_14416_b200 import binding as B
from paper_2010_14416_b200 import workloads as W


def main(names):
    ok = True
    for name in names:
        if name.startswith("sweep_"):            # config 5: sweep_0.1M ... sweep_50M
            w = W.config5(name[len("sweep_"):])
        else:
            w = {"config1": W.config1, "config2": W.config2, "config3": W.config3, "config4": W.config4}[name]()
        t0 = time.time()
        m = B.SweMesh.from_workload(w).bind_device()
        m.set_state(w.h, w.hu, w.hv)
        m.run(w.nsteps)
        hg, hug, hvg, tg, dtg = m.get_state()
        t_gpu = time.time() - t0
        t0 = time.time()
        o = OracleSolver.from_workload(w)
        done = o.run(w.nsteps)
        ho, huo, hvo, to, dto = o.get_state()
        t_cpu = time.time() - t0

        def dev(a, b):      # deviation in units of the bar: |a-b| / (1e-10 + 1e-10 |b|)
            return float(np.max(np.abs(a - b) / (1e-10 + 1e-10 * np.abs(b))))

        mask_equal = bool(np.array_equal(hg <= w.h_dry, ho <= w.h_dry))
        devs = dict(h=dev(hg, ho), hu=dev(hug, huo), hv=dev(hvg, hvo))
        rel_t, rel_dt = abs(tg - to) / abs(to), abs(dtg - dto) / abs(dto)
        good = done == w.nsteps and mask_equal and max(devs.values()) <= 1.0 and rel_t <= 1e-12 and rel_dt <= 1e-12
        ok &= good
        st = m.get_stats()
        print(f"{name}: {w.ncells} cells x {w.nsteps} steps  {'PASS' if good else 'FAIL'}\n"
              f"  max deviation / bar: h {devs['h']:.3e}  hu {devs['hu']:.3e}  hv {devs['hv']:.3e}\n"
              f"  |dt| rel {rel_t:.2e}  |ddt| rel {rel_dt:.2e}  dry mask identical: {mask_equal}  "
              f"dry cells {int(st['n_dry'])}  clamps {int(st['n_clamped'])}\n"
              f"  wall time incl. set-up: GPU path {t_gpu:.1f} s, oracle ({o.threads} threads) {t_cpu:.1f} s", flush=True)
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:] or ["config3", "config4"]))
