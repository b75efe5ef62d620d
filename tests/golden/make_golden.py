"""Writes tests/golden/ring_chain.txt and small_graphs.txt from tests/closed_forms.py (scipy Bessel
sums and brute-force quadrature).  Calls neither the CUDA path nor oracle/.  The values restate
SURVEY.md Appendix A (computed there the same way); test_oracle_equilibrium.py re-derives them live.
Run:  python tests/golden/make_golden.py"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
import closed_forms as CF  # noqa: E402

with open(os.path.join(HERE, "ring_chain.txt"), "w") as f:
    f.write("# periodic ring (Z ~ sum_n I_n(beta)^N) and open chain (tree) closed forms; SURVEY.md Appendix A,\n"
            "# BASELINE.json north_star 'exact ring closed form'.  columns: kind N T e=E/N <m^2>\n")
    for N in (8, 16, 64, 256):
        for T in (0.5, 1.0, 2.0, 4.0):
            e, m2 = CF.ring(N, 1 / T)
            f.write(f"ring {N} {T} {e:.10f} {m2:.10f}\n")
    for N in (16, 256):
        for T in (0.5, 1.0, 2.0, 4.0):
            e, m2 = CF.chain(N, 1 / T)
            f.write(f"chain {N} {T} {e:.10f} {m2:.10f}\n")

with open(os.path.join(HERE, "small_graphs.txt"), "w") as f:
    f.write("# brute-force quadrature (periodic trapezoid, 64 points per free angle) on 3- and 4-site graphs;\n"
            "# SURVEY.md Appendix A.  columns: graph beta <E> VarE <|m|> <m^2> <m^4> U4\n")
    for name, (N, edges) in CF.SMALL_GRAPHS.items():
        for beta in (0.5, 1.0, 2.0):
            q = CF.quadrature(N, edges, beta)
            f.write(f"{name} {beta} {q['E']:.10f} {q['varE']:.10f} {q['absm']:.10f} {q['m2']:.10f} {q['m4']:.10f} "
                    f"{q['m4'] / q['m2'] ** 2 - 1:.10f}\n")
