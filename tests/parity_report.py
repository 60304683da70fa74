"""Turns the JSON-lines records the parity tests append (gpurun_out/parity_records.jsonl, see
parity_util.record_parity) into the tracked summary profiles/parity_r<round>.json.

    python tests/parity_report.py [--round 2] [--records gpurun_out/parity_records.jsonl]

Keeps the LAST record of every test label (a re-run supersedes an earlier one), sorted by margin, and
states the worst margin to the north_star tolerance.  Reads only what the tests wrote; computes
nothing about the method itself.
"""
import argparse
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--round", type=int, default=2)
    ap.add_argument("--records", default=os.path.join(ROOT, "gpurun_out", "parity_records.jsonl"))
    ap.add_argument("--commit", default="", help="commit the records were measured on")
    args = ap.parse_args()
    last = {}
    with open(args.records) as f:
        for line in f:
            line = line.strip()
            if line:
                r = json.loads(line)
                last[r["what"]] = r
    def limit(r):
        # a record that carries the bf16 rounding floor of its own (heavy-tailed) output is checked
        # against max(tolerance, floor + 5e-2), as its test does (test_saturated_gates_parity)
        fl = r.get("bf16_output_rounding_floor_max_over_rms")
        return r["tol_max_over_rms"] if fl is None else max(r["tol_max_over_rms"], fl + 5e-2)

    for r in last.values():
        r["limit_max_over_rms"] = limit(r)
        r["margin_max_over_rms"] = 1.0 - r["max_over_rms"] / r["limit_max_over_rms"]

    def section(r):
        w = r["what"]
        if w.startswith("backward"):
            return "backward"            # gradients: north_star states no tolerance; held to the forward's
        if w.startswith("cfg"):
            return "baseline_configs"    # BASELINE.json configs 0-4, the tolerances north_star binds
        if "bf16_output_rounding_floor_max_over_rms" in r or "precondition" in w:
            return "stress"
        return "other_forward"

    key = lambda r: min(r["margin_rel_fro"], r["margin_max_over_rms"])
    groups = {}
    for r in last.values():
        groups.setdefault(section(r), []).append(r)
    for g in groups.values():
        g.sort(key=key)
    pick = lambda r: {k: r[k] for k in ("what", "rel_fro", "max_over_rms", "limit_max_over_rms",
                                        "margin_rel_fro", "margin_max_over_rms")}
    recs = sorted(last.values(), key=key)
    worst = groups.get("baseline_configs", recs)[0] if recs else None
    out = {
        "tolerances": "north_star: bf16 rel-Frobenius <= 1e-2 and max-abs <= 5e-2 * rms(out); fp32 mode rel-Frobenius <= 1e-5",
        "margin": "1 - measured / limit (0.10 = 10 % under the limit); limit_max_over_rms is the tolerance, except "
                  "for records that carry bf16_output_rounding_floor_max_over_rms (output so heavy-tailed that "
                  "rounding the exact result to bf16 already exceeds 5e-2 * rms): max(tolerance, floor + 5e-2)",
        "measured_on_commit": args.commit,
        "n_records": len(recs),
        "worst": None if worst is None else pick(worst),
        "worst_per_section": {name: pick(g[0]) for name, g in sorted(groups.items())},
        "records": {name: g for name, g in sorted(groups.items())},
    }
    path = os.path.join(ROOT, "profiles", f"parity_r{args.round}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(f"{path}: {len(recs)} records; worst margin: {None if worst is None else worst['what']}")


if __name__ == "__main__":
    main()
