"""Count the algorithmic FP64 operations per cell update of the ORACLE's time step.

Builds oracle/opcount/libmmo_counted.so (the oracle's .c files with `double` replaced by the
counting type of opcount.hpp), runs a few steps of the crossed-jet and Sod workloads through it
and writes tests/golden/oracle_opcount.txt.  Calls only oracle/ and the input generators.

    python oracle/opcount/count_flops.py
"""
import ctypes as C
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
ROOT = HERE.parents[1]
sys.path.insert(0, str(ROOT))

import mm_workloads as wl  # noqa: E402
from oracle import mmo  # noqa: E402


def build():
    out = HERE / "libmmo_counted.so"
    subprocess.run(["g++", "-std=c++17", "-O1", "-fPIC", "-shared", "-fpermissive", "-w", "-o", str(out),
                    str(HERE / "mmo_counted.cpp")], check=True, cwd=HERE)
    return out


def main():
    L = mmo.bind(C.CDLL(str(build())))
    L.mmo_opcount_get.restype = C.c_longlong
    mmo._lib = L                                     # this process drives the counted build only

    def count(prob, nsteps, cfl, warm=0):
        s = mmo.Solver(prob["system"], prob["nx"], prob["ny"], extent=prob["extent"],
                       collision=prob["collision"], bcs=prob["bcs"], nthreads=1, **prob["options"])
        s.set_state_prim(prob["W0"])
        if warm:
            s.step(warm, cfl)
        L.mmo_opcount_reset()
        s.step(nsteps, cfl)
        return L.mmo_opcount_get() / (prob["nx"] * prob["ny"] * nsteps)

    lines = ["# Algorithmic FP64 operations per cell update of the oracle's time step, counted by",
             "# oracle/opcount/count_flops.py (each + - * / sqrt exp pow = 1; comparisons, fabs, copies = 0).",
             "# Includes the ghost-cell cons->prim and wave speeds and the tile-independent (N+1)/N interfaces.",
             "# name  ops_per_cell_update  workload"]
    n = 96
    a = count(wl.crossed_jets(n, Kn=0.1, perturb=0.01), 4, 0.4, warm=60)
    lines.append(f"flops_per_cell_update_14 {a:.1f} crossed_jets({n}, Kn=0.1, perturb=0.01), minmod shared + HLL, "
                 f"4 CFL steps after 60 warm-up steps")
    b = count(wl.crossed_jets(n, Kn=None, perturb=0.01), 4, 0.4, warm=60)
    lines.append(f"flops_per_cell_update_14_collisionless {b:.1f} same, tau = inf")
    c = count(wl.sod14(512, 4, Kn=0.01), 4, 0.5, warm=20)
    lines.append(f"flops_per_cell_update_14_sod {c:.1f} sod14(512, 4, Kn=0.01), per-variable minmod + HLL")
    d = count(wl.sod5(1000, Kn=0.01), 4, 0.5, warm=20)
    lines.append(f"flops_per_cell_update_5 {d:.1f} sod5(1000, Kn=0.01), minmod + HLL")
    out = ROOT / "tests" / "golden" / "oracle_opcount.txt"
    out.write_text("\n".join(lines) + "\n")
    print(out.read_text())


if __name__ == "__main__":
    main()
