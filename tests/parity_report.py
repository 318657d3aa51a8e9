"""Runs the GPU parity tests and writes their records as a Markdown report (profiles/r02_parity.md).

    python tests/parity_report.py [out.md]

Calls only the tests: every number comes from the `PARITY` records that tests/test_gpu_parity.py appends to the file
named by WPCD_PARITY_REPORT -- worst error / tolerance per comparison, the histogram of the plain relative errors
(SURVEY.md section 8(c)9), and the first-bin comparison against the long-double build of the oracle's rule."""
import json
import os
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def main():
    out = sys.argv[1] if len(sys.argv) > 1 else os.path.join(ROOT, "profiles", "r02_parity.md")
    with tempfile.NamedTemporaryFile(suffix=".jsonl", delete=False) as f:
        rec_path = f.name
    env = dict(os.environ, WPCD_PARITY_REPORT=rec_path)
    cmd = [sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_parity.py"), "-m", "gpu", "-q", "-p", "no:cacheprovider"]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True)
    tail = r.stdout.strip().splitlines()[-1] if r.stdout.strip() else ""
    recs = [json.loads(line) for line in open(rec_path) if line.strip()]
    os.unlink(rec_path)
    lines = ["# r02 -- value parity of the CUDA path against the CPU oracle (one B200)", "",
             "Command: `python tests/parity_report.py` (runs `pytest tests/test_gpu_parity.py -m gpu`; pytest said: `" + tail + "`).", "",
             "Tolerance of every comparison: |v_gpu - v_oracle| <= 1e-11 max(|v|, A_e) + 1e-13 V (A_e: absolute term sum, V: largest",
             "|v| of the matrix; DESIGN.md R9).  `worst err/tol` is the largest ratio seen.  `well` = entries with A_e < 10 |v| (no",
             "cancellation between the (k,l1,l1') terms); an entry of that kind beyond 1e-11 relative fails the test unless its error is",
             "below the absolute floor 1e-13 V (sliver elements: a tiny support, not a cancellation, makes |v| small).", "",
             "Histogram columns: number of entries with plain relative error in [0,1e-15), [1e-15,1e-14), [1e-14,1e-13), [1e-13,1e-12),",
             "[1e-12,1e-11), [1e-11,1e-10), [1e-10,1e-9), [1e-9,1e-6), [1e-6,1e-3), [1e-3,inf).", "",
             "| test | lattice | n | rule | entries | well | worst err/tol | worst rel (well) | worst rel (all) | histogram (all) | histogram (well) |",
             "|---|---|---|---|---|---|---|---|---|---|---|"]
    for x in recs:
        if "hist_rel_err" not in x:
            continue
        lines.append("| {} | {}x{} | {} | {} | {} | {} | {:.2e} | {:.1e} | {:.1e} | {} | {} |".format(
            x["test"], x.get("n_p"), x.get("n_q"), x.get("n_quad"), {0: "R", 1: "RS", 2: "RA"}.get(x.get("rule"), "R"), x["entries"],
            x["well_conditioned"], x["worst_err_over_tol"], x["worst_rel_err_well_conditioned"], x["worst_rel_err"],
            " ".join(str(v) for v in x["hist_rel_err"]), " ".join(str(v) for v in x["hist_rel_err_well_conditioned"])))
    lines += ["", "## First-bin cells against the long-double evaluation of the same rule", "",
              "Entries of cells touching p = 0 or p' = 0 with l, l' >= 2 (SURVEY 8(c)8); errors in units of eps A_e, eps = 2^-53.", "",
              "| J^pi | N | entries | median A_e/|v| | max A_e/|v| | rms err CUDA | rms err FP64 oracle | max err CUDA | max err FP64 oracle |",
              "|---|---|---|---|---|---|---|---|---|"]
    for x in recs:
        if x.get("test") != "first_bin_extended":
            continue
        lines.append("| {}/2{} | {} | {} | {:.1e} | {:.1e} | {:.2f} | {:.2f} | {:.1f} | {:.1f} |".format(
            x["J2"], "+" if x["parity"] > 0 else "-", x["n_bins"], x["entries"], x["median_cond"], x["max_cond"], x["rms_err_gpu_eps_Ae"],
            x["rms_err_oracle64_eps_Ae"], x["max_err_gpu_eps_Ae"], x["max_err_oracle64_eps_Ae"]))
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
    print(out, tail)
    return r.returncode


if __name__ == "__main__":
    sys.exit(main())
