"""Turn the records the full-size parity tests write (tests/test_gpu_fullsize.py -> gpurun_out/parity_fullsize.jsonl) into
the markdown table kept under profiles/:

    python -m paper_2508_05343_b200.parity_table gpurun_out/parity_fullsize.jsonl > profiles/r03_parity_fullsize.md

Formatting only: no arithmetic of the method, nothing from oracle/.  When a case occurs more than once in the file (the
file is appended to by every run) the last record wins."""
from __future__ import annotations

import json
import sys


def main(path: str) -> None:
    recs = {}
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line:
                r = json.loads(line)
                recs[r["case"]] = r
    print("# Full-size parity against the oracle (every pixel, every gradient tensor, unmasked)\n")
    print("Written by `python -m paper_2508_05343_b200.parity_table %s` from the records of" % path)
    print("`python -m pytest tests/test_gpu_fullsize.py -m gpu` on one B200.  Bars: image / final T 1e-4, gradients 1e-3")
    print("(inf-norm relative, per tensor), last contributor exact, `violations` 0.\n")
    print("| case | N | K | D | undecidable px (of) | image max err | final T max err | worst gradient tensor (rel inf) | worst element (rel) |")
    print("|---|---|---|---|---|---|---|---|---|")
    for case in sorted(recs):
        r = recs[case]
        wn = max(r["grad_rel_inf"], key=lambda k: r["grad_rel_inf"][k])
        en = max(r["grad_rel_elementwise"], key=lambda k: r["grad_rel_elementwise"][k])
        print("| %s | %d | %d | %d | %d (%d) | %.2e | %.2e | %s %.2e | %s %.2e |" % (
            case, r["N"], r["K"], r["D"], r["undecidable"], r["pixels"], r["image_max_err"], r["final_T_max_err"],
            wn, r["grad_rel_inf"][wn], en, r["grad_rel_elementwise"][en]))


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "gpurun_out/parity_fullsize.jsonl")
