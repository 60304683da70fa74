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
    recs = sorted(last.values(), key=lambda r: min(r["margin_rel_fro"], r["margin_max_over_rms"]))
    worst = recs[0] if recs else None
    out = {
        "tolerances": "north_star: bf16 rel-Frobenius <= 1e-2 and max-abs <= 5e-2 * rms(out); fp32 mode rel-Frobenius <= 1e-5",
        "margin": "1 - measured / tolerance (0.10 = 10 % under the limit)",
        "measured_on_commit": args.commit,
        "n_records": len(recs),
        "worst": None if worst is None else {k: worst[k] for k in ("what", "rel_fro", "max_over_rms", "margin_rel_fro", "margin_max_over_rms")},
        "records": recs,
    }
    path = os.path.join(ROOT, "profiles", f"parity_r{args.round}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(f"{path}: {len(recs)} records; worst margin: {None if worst is None else worst['what']}")


if __name__ == "__main__":
    main()
