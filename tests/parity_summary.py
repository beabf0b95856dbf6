"""Turn the parity record the GPU suite wrote (tests/_util.record_parity, JSON lines) into the
markdown table committed under profiles/.

    python tests/parity_summary.py gpurun_out/parity_record.jsonl > profiles/parity_r02.md
"""
import json
import sys


def main(path):
    rows = [json.loads(l) for l in open(path) if l.strip()]
    f = lambda v: "" if v is None else (f"{v:.2e}" if isinstance(v, float) else str(v))
    print("# Measured parity: CUDA path against the CPU oracle\n")
    print("Written by `tests/parity_summary.py` from the record of one `pytest tests -m gpu` run on a B200 "
          "(`profiles/parity_r02.jsonl`, one line per comparison).  Norm: max |gpu - oracle| over all components "
          "and entries of the vector field / max |oracle| (DESIGN.md A21); `M / change` divides by "
          "max |oracle - M at t = 0| instead (how far M moved).  The bar is 1e-9 (north_star).\n")
    print("| test | config | shape | steps | path | err E | err H | err M | M / change | LLG iterations (gpu = oracle) |")
    print("|---|---|---|---:|---|---:|---:|---:|---:|---|")
    for r in rows:
        if "err_E" not in r:
            continue
        it = ""
        if "iters" in r:
            it = str(r["iters"]) + (" = " + str(r["iters_oracle"]) if "iters_oracle" in r else "")
        print(f"| {r['test']} | {r['config']} | {'x'.join(map(str, r['shape']))} | {r['steps']} | {r.get('path', '')}"
              f"{' (merged H)' if r.get('merged_h') else ''} | {f(r.get('err_E'))} | {f(r.get('err_H'))} | "
              f"{f(r.get('err_M'))} | {f(r.get('err_M_over_change'))} | {it} |")
    extra = [r for r in rows if "err_E" not in r]
    if extra:
        print("\nOther records:\n")
        for r in extra:
            print("- " + ", ".join(f"{k} = {f(v)}" for k, v in r.items()))
    worst = {g: max((r.get("err_" + g) or 0.0) for r in rows if r.get("steps") == 100) for g in "EHM"}
    print(f"\nWorst after 100 steps: E {worst['E']:.2e}, H {worst['H']:.2e}, M {worst['M']:.2e}.")


if __name__ == "__main__":
    main(sys.argv[1])
