"""Count the algorithmic operations per cell update with the oracle (TEST INFRASTRUCTURE ONLY).

Builds oracle/libflopcount.so (flop_count.cpp = hydro_oracle.cpp instantiated with a counting
scalar) and writes oracle/flops_per_cell.json, which bench.py's roofline reads.  Calls only oracle/
and the seeded input generators.  Run: python -m oracle.count_flops
"""
import ctypes as C
import json
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
LIB = os.path.join(HERE, "libflopcount.so")
SRC = os.path.join(HERE, "flop_count.cpp")


LIB_RTVD = os.path.join(HERE, "libflopcount_rtvd.so")
SRC_RTVD = os.path.join(HERE, "flop_count_rtvd.cpp")


def build_rtvd():
    deps = [SRC_RTVD, os.path.join(HERE, "rtvd_oracle.cpp"), os.path.join(HERE, "flop_scalar.h")]
    if not os.path.exists(LIB_RTVD) or any(os.path.getmtime(d) > os.path.getmtime(LIB_RTVD) for d in deps):
        subprocess.run(["g++", "-std=c++17", "-O1", "-shared", "-fPIC", "-o", LIB_RTVD, SRC_RTVD], check=True, cwd=HERE)
    return LIB_RTVD


def build_split(name):
    lib_, src = os.path.join(HERE, "libflopcount_%s.so" % name), os.path.join(HERE, "flop_count_%s.cpp" % name)
    deps = [src, os.path.join(HERE, name + "_oracle.cpp"), os.path.join(HERE, "flop_scalar.h")]
    if not os.path.exists(lib_) or any(os.path.getmtime(d) > os.path.getmtime(lib_) for d in deps):
        subprocess.run(["g++", "-std=c++17", "-O1", "-shared", "-fPIC", "-o", lib_, src], check=True, cwd=HERE)
    return lib_


def count_waf(G, dt, dh, gamma, order=0):
    L = C.CDLL(build_split("waf"))
    G = np.ascontiguousarray(G, np.float64)
    Ng, S = G.shape[0], G.shape[2]
    c = np.zeros(7, np.int64)
    L.oracle_waf_count_ops.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                       C.POINTER(C.c_longlong)]
    L.oracle_waf_count_ops(G.ctypes.data_as(C.POINTER(C.c_double)), Ng, (S - 16) // 2, dt, dh, gamma, order,
                           c.ctypes.data_as(C.POINTER(C.c_longlong)))
    cells = Ng * 16 ** 3
    per = {n: float(v) / cells for n, v in zip(("add", "mul", "div", "sqrt", "pow", "cmp", "abs"), c)}
    per["flops_per_cell"] = per["add"] + per["mul"] + per["div"] + per["sqrt"] + per["pow"]
    return per


def count_rtvd(G, dt, dh, gamma, order=0):
    L = C.CDLL(build_rtvd())
    G = np.ascontiguousarray(G, np.float64)
    Ng, S = G.shape[0], G.shape[2]
    c = np.zeros(7, np.int64)
    L.oracle_rtvd_count_ops.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                        C.POINTER(C.c_longlong)]
    L.oracle_rtvd_count_ops(G.ctypes.data_as(C.POINTER(C.c_double)), Ng, (S - 16) // 2, dt, dh, gamma, order,
                            c.ctypes.data_as(C.POINTER(C.c_longlong)))
    cells = Ng * 16 ** 3
    per = {n: float(v) / cells for n, v in zip(("add", "mul", "div", "sqrt", "pow", "cmp", "abs"), c)}
    per["flops_per_cell"] = per["add"] + per["mul"] + per["div"] + per["sqrt"] + per["pow"]
    return per


def build():
    deps = [SRC, os.path.join(HERE, "hydro_oracle.cpp"), os.path.join(HERE, "flop_scalar.h")]
    if not os.path.exists(LIB) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in deps):
        subprocess.run(["g++", "-std=c++17", "-O1", "-shared", "-fPIC", "-o", LIB, SRC], check=True, cwd=HERE)
    return LIB


def count(G, dt, dh, gamma, scheme, riemann, limiter, recon=0, char_limit=0, want_flux=1):
    L = C.CDLL(build())
    G = np.ascontiguousarray(G, np.float64)
    Ng, S = G.shape[0], G.shape[2]
    g = (S - 16) // 2
    c = np.zeros(8, np.int64)
    L.oracle_count_ops.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                   C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_longlong)]
    L.oracle_count_ops(G.ctypes.data_as(C.POINTER(C.c_double)), Ng, g, dt, dh, gamma, scheme, riemann, limiter, recon,
                       char_limit, want_flux, c.ctypes.data_as(C.POINTER(C.c_longlong)))
    cells = Ng * 16 ** 3
    names = ("add", "mul", "div", "sqrt", "pow", "cmp", "abs", "riemann_solves")
    per = {n: float(v) / cells for n, v in zip(names, c)}
    per["flops_per_cell"] = per["add"] + per["mul"] + per["div"] + per["sqrt"] + per["pow"]
    return per


def main():
    from oracle import oracle as O
    from paper_1103_3373_b200 import workloads as wl
    MHM, VL, CTU = 0, 1, 2
    EXACT, HLLE, HLLC, ROE = 0, 1, 2, 3
    gamma, dh = 5.0 / 3.0, 1.0
    out = {"_about": "algorithmic operations per interior cell update, counted on the CPU oracle (oracle/flop_count.cpp) over the oracle's regions; input: first 8 groups of workloads.amr_batch(seed=0), dt = CFL*dh/hydro_dt.  CTU and MHM: the oracle's regions are within 1.3 % of the minimal per-group multiplicities of SURVEY.md 8(a) (7.22 vs 7.17 and 3.19 vs 3.19 Riemann solves per cell).  VL: the oracle's predictor region is a box, not the minimal plus: 9.34 / 11.34 solves per cell (PLM / PPM) against the minimal 8.72 / 9.89, i.e. the VL counts are 7 % / 15 % above what the method must compute and roofline fractions quoted from them are flattering by about half of that",
           "_minimal_riemann_per_cell": {"ctu": 7.17, "mhm": 3.19, "vl_plm": 8.72, "vl_ppm": 9.89, "source": "SURVEY.md 8(a)"},
           "_flop_rule": "add, sub, mul, div, sqrt, pow = 1 each; compare/abs/min/max/select/negate = 0"}
    cases = {
        "ctu_plm_roe_vanleer_g3": (CTU, ROE, 1, 0, 3, 0.5),
        "ctu_plm_hllc_vanleer_g2": (CTU, HLLC, 1, 0, 2, 0.5),
        "ctu_plm_hlle_vanleer_g2": (CTU, HLLE, 1, 0, 2, 0.5),
        "ctu_ppm_roe_vanleer_g3": (CTU, ROE, 1, 1, 3, 0.5),
        "ctu_ppm_exact_vanleer_g3": (CTU, EXACT, 1, 1, 3, 0.5),
        "mhm_plm_roe_vanleer_g2": (MHM, ROE, 1, 0, 2, 0.3),
        "mhm_ppm_roe_vanleer_g3": (MHM, ROE, 1, 1, 3, 0.3),
        "vl_plm_roe_vanleer_g3": (VL, ROE, 1, 0, 3, 0.3),
        "vl_ppm_roe_vanleer_g4": (VL, ROE, 1, 1, 4, 0.3),
    }
    for name, (scheme, riemann, limiter, recon, g, cfl) in cases.items():
        G = wl.amr_batch(8, g=g, gamma=gamma, seed=0, dtype="float64").numpy()
        dt = cfl * dh / O.hydro_dt(G, gamma, 0)
        out[name] = count(G, dt, dh, gamma, scheme, riemann, limiter, recon)
        print(name, {k: round(v, 1) for k, v in out[name].items()})
    G = wl.amr_batch(8, g=3, gamma=gamma, seed=0, dtype="float64").numpy()
    out["rtvd_g3"] = count_rtvd(G, 0.3 * dh / O.hydro_dt(G, gamma, 0), dh, gamma, 0)
    out["rtvd_g3"]["_note"] = ("three split sweeps over the oracle's ranges (484 + 352 + 256 pencils of 22 cells per group): "
                               "5.9 cell-sweeps per interior cell update")
    print("rtvd_g3", {k: round(v, 1) for k, v in out["rtvd_g3"].items() if k != "_note"})
    out["waf_g3"] = count_waf(G, 0.3 * dh / O.hydro_dt(G, gamma, 0), dh, gamma, 0)
    out["waf_g3"]["_note"] = "three split WAF sweeps over the oracle's ranges (the 22-cell pencils of the RTVD batches): 5.9 cell-sweeps per interior cell update"
    print("waf_g3", {k: round(v, 1) for k, v in out["waf_g3"].items() if k != "_note"})
    with open(os.path.join(HERE, "flops_per_cell.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
