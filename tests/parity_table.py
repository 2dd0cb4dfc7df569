"""Markdown summary of the parity-error CSV the GPU tests write (`FRB_PARITY_CSV`, default gpurun_out/parity_errors.csv):

  python tests/parity_table.py profiles/r02_parity_errors.csv

One row per (test, precision): comparisons, worst achieved error, comparisons above the north_star tolerance and, among those, the
worst error in units of 2^-24 * amp (reading R23 asserts 3).  Not a test (pytest collects test_*.py only).
"""
import csv
import re
import sys


def main(path):
    rows = list(csv.DictReader(open(path)))
    agg = {}
    for r in rows:
        key = (re.sub(r"\[.*", "", r["test"]), r["prec"])
        a = agg.setdefault(key, dict(n=0, worst=0.0, above=0, ratio=0.0))
        err, tol, amp = float(r["achieved_rel_err"]), float(r["north_star_tol"]), float(r["amp"])
        a["n"] += 1
        a["worst"] = max(a["worst"], err)
        if err > tol:
            a["above"] += 1
            a["ratio"] = max(a["ratio"], err / (2.0 ** -24 * amp))
    print("| test | precision | comparisons | worst achieved error | comparisons above the north_star tolerance | worst err / (2^-24 amp) among those |")
    print("|---|---|---|---|---|---|")
    for (t, p), a in sorted(agg.items()):
        print("| `%s` | %s | %d | %.2e | %d | %s |" % (t, p, a["n"], a["worst"], a["above"], ("%.2f" % a["ratio"]) if a["above"] else "-"))
    for p in ("f64", "f32"):
        sel = [r for r in rows if r["prec"] == p]
        if not sel:
            continue
        err = [float(r["achieved_rel_err"]) for r in sel]
        ok = sum(float(r["achieved_rel_err"]) <= float(r["north_star_tol"]) for r in sel)
        print("")
        print("%s: %d comparisons, %d (%.0f %%) within the north_star tolerance, worst achieved error %.2e; every one within the asserted tolerance: %s."
              % (p.upper(), len(sel), ok, 100.0 * ok / len(sel), max(err),
                 all(float(r["achieved_rel_err"]) <= float(r["asserted_tol"]) for r in sel)))


if __name__ == "__main__":
    main(sys.argv[1])
