"""Exact FP64 operation counts of the method, from an op-counting build of the oracle (MEASUREMENT ONLY).

    python -m oracle.count_ops            # prints a markdown table (committed as profiles/r2_oracle_flops.md)

Builds oracle/tfo.cpp with -DTFO_COUNT_OPS (oracle/opcount.h: `double` becomes a counting scalar) into
liboracle_tfo_count.so and counts, with one thread: the point functions (one Maxwell flux, one AUSM+-up flux, one
source, one U(P)), the gradient + limiter per cell, the residual per cell and Algorithm 1's residual + Jacobian per
cell -- the oracle follows Alg. 1 literally (nFaces x (1 + 18) full 18-row flux evaluations from each side).  From the
point-function counts it composes the algorithmic count of the CUDA path's design (block-diagonal flux
Jacobian, own side only: 9 Maxwell + 2 x 6 AUSM evaluations per cell-face).  Calls only oracle/.
"""
import ctypes as C
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
SO = os.path.join(HERE, "liboracle_tfo_count.so")
NAMES = ["add", "mul", "div", "sqrt", "pow", "cmp", "sign"]


def build():
    src = os.path.join(HERE, "tfo.cpp")
    cmd = ["g++", "-std=c++17", "-O1", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-DTFO_COUNT_OPS",
           "-o", SO, src]
    subprocess.run(cmd, check=True, cwd=HERE)
    return SO


def main():
    build()
    from oracle import binding as B
    from paper_1809_02532_b200 import workloads as W
    # the binding, pointed at the counting library
    B._SO = SO
    B._lib = None
    B.build = lambda force=False: SO
    L = B.lib()
    L.tfo_opcount_get.argtypes = [C.POINTER(C.c_int64)]
    L.tfo_opcount_reset.argtypes = []
    B.set_num_threads(1)

    def counted(fn):
        L.tfo_opcount_reset()
        fn()
        out = (C.c_int64 * 8)()
        L.tfo_opcount_get(out)
        return np.array(list(out)[:7], dtype=np.int64)

    flops = lambda c: int(c[:5].sum())          # add + mul + div + sqrt + pow, one flop each
    ph = B.physics_c()
    nu = B.default_numerics(ph)
    rng = np.random.default_rng(0)
    P = np.abs(rng.normal(size=(2, 18))) + 0.5
    P[:, 9] /= 25.0
    rows = []
    point = {}
    for name, fn in (("Maxwell flux, one evaluation (8 rows)", lambda: B.flux_maxwell(ph, P[0, :8], P[1, :8], 0.6, 0.8)),
                     ("AUSM+-up flux, one species, one evaluation (5 rows)",
                      lambda: B.flux_ausm(ph, nu, 0, P[0, [8, 10, 11, 12, 16]], P[1, [8, 10, 11, 12, 16]], 0.6, 0.8)),
                     ("full face flux (Maxwell + 2 species)", lambda: B.flux_face(ph, nu, P[0], P[1], 0.6, 0.8)),
                     ("source S(P), one evaluation", lambda: B.source(ph, P[0])),
                     ("U(P), one evaluation", lambda: B.cons(ph, P[0]))):
        c = counted(fn)
        point[name] = c
        rows.append((name, c, None))
    mxw, ausm, src_c, cons_c = (point[k] for k in list(point)[:2] + list(point)[3:5])

    out = ["# Exact FP64 operation counts (op-counting build of the oracle)", "",
           "Command: `python -m oracle.count_ops` (builds `oracle/tfo.cpp` with `-DTFO_COUNT_OPS`; one thread; calls only",
           "`oracle/`).  flops = add + mul + div + sqrt + pow, one each (SURVEY 8(d)); comparisons and sign operations are",
           "listed but not counted as flops.", "",
           "| quantity | " + " | ".join(NAMES) + " | flops |", "|---|" + "---|" * 8]
    for name, c, _ in rows:
        out.append(f"| {name} | " + " | ".join(str(int(x)) for x in c) + f" | {flops(c)} |")

    for wname, mi in (("triangles (Delaunay, 2 500 cells, config 4's recipe)",
                       W.delaunay_mesh(51, 26, *W.GEM_DOMAIN, jitter=0.3, seed=2, shuffle_cells=True)),
                      ("quadrilaterals (50 x 50, periodic, q1's recipe)", W.quad_mesh(50, 50, -12.8, 12.8, -12.8, 12.8))):
        o = B.OracleMesh.from_input(mi)
        nc = o.n_cells
        st = W.gem_state(mi.centroids()) + rng.uniform(-1e-3, 1e-3, (nc, 18))
        g = counted(lambda: B.gradients(o, nu, st))
        r = counted(lambda: B.assemble(o, ph, nu, st, jacobian=False))
        j = counted(lambda: B.assemble(o, ph, nu, st, jacobian=True))
        nf_c = o.max_faces if "quad" in wname else 3
        nst = o.n_stencil / nc
        out += ["", f"### {wname}: per cell (averages over {nc} cells; {nst:.1f} stencil entries per cell)", "",
                "| step | " + " | ".join(NAMES) + " | flops per cell |", "|---|" + "---|" * 8]
        for name, c in (("a2 gradient + limiter (tfo_gradients)", g),
                        ("residual only: a2 + fluxes of the cell's faces + source + BDF2", r),
                        ("Algorithm 1 as the oracle runs it: residual + Jacobian (every face from both cells, 1 + 2 x 18 full evaluations per face visit)", j)):
            out.append(f"| {name} | " + " | ".join(f"{x / nc:.0f}" for x in c) + f" | {flops(c) / nc:.0f} |")
        # the CUDA path's design: per cell-face 1 base + 8 perturbed Maxwell evaluations and, per species, 1 base + 5
        # perturbed AUSM evaluations (own side only); 18 perturbed sources (each group's rows only: counted in full
        # here, an upper bound); differencing 2 flops per Jacobian entry produced (114 per face + 324 diagonal)
        design = nf_c * (9 * mxw + 12 * ausm) + 19 * src_c + 3 * cons_c
        diff = 2 * (nf_c * 114 + 324)
        tot = flops(g) / nc + flops(design) + diff
        out += ["", f"Algorithmic count of the CUDA path's design on this mesh: gradient + limiter {flops(g) / nc:.0f} + "
                f"{nf_c} faces x (9 Maxwell + 12 AUSM evaluations) + 19 sources + 3 U(P) = {flops(design)} + differencing "
                f"{diff} = **{tot:.0f} flops per cell**."]
    print("\n".join(out))


if __name__ == "__main__":
    main()
