"""Writes tests/golden/scaling_start_N36.txt: the start vector of "config 2'" (the paper's own parameter set, PAPER.md L135,
L143, L188, L364), used by workloads.scaling_start_coefficients, bench.py --config 2 and the tests.

    python tests/golden/make_scaling_start.py

Calls only oracle/ (through tests/scaling_setup.py, where the guess is defined: the paper's asymptotic forms eq.(16)-(19)
sampled at the mapped Chebyshev roots, fn.9, projected on T_j with the oracle's tables, a_0 shifted so that
Z(x_Z) = 0.256).  Nothing here comes from the CUDA path.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))                     # tests/
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))    # repo root


def main():
    import scaling_setup as S
    from oracle.oracle import Oracle, make_params
    orc = Oracle()
    p = make_params(S.N, S.N_R, S.N_THETA, S.EPS2, S.L2, 0.0, S.L2, n_ir=S.N_IR)
    c = S.start_coefficients(orc, p)
    with open(os.path.join(HERE, "scaling_start_N36.txt"), "w") as f:
        f.write("# start vector of config 2' (PAPER.md L135, L364; DESIGN.md reading A17): c = (a_0..a_35, b_0..b_35),\n"
                "# written by tests/golden/make_scaling_start.py from oracle/ only (tests/scaling_setup.start_coefficients)\n")
        for v in c:
            f.write(f"{float(v)!r}\n")


if __name__ == "__main__":
    main()
