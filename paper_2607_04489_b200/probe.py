"""Machine probes of libeiger (eiger_probe): prints one JSON line per measured building-block rate.

    python -m paper_2607_04489_b200.probe [--quick]

The numbers behind DESIGN.md section 5 ("machine facts") and the selector's thresholds; the summary
of a run on the B200 is kept in profiles/r2_probe.md.
"""
from __future__ import annotations

import json
import sys

import paper_2607_04489_b200 as eiger


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    quick = "--quick" in argv
    plan = [("read_ldg", 4096, 0, "GB/s"), ("read_bulk", 4096, 8192, "GB/s"), ("read_bulk", 4096, 16384, "GB/s"),
            ("read_bulk", 4096, 32768, "GB/s")]
    for mode in ("dsmem_red", "dsmem_atom", "dsmem_cas", "dsmem_st"):
        for c in (1, 2, 4, 8, 16):
            for slots in ((8192,) if quick else (1024, 8192)):
                plan.append((mode, c, slots, "G rows/s"))
    for c in (2, 4, 8, 16):
        for chunk in (1024, 4096):
            plan.append(("dsmem_bulk", c, chunk, "GB/s"))
    for chunk in (128, 256, 512, 1024, 4096):
        plan.append(("store_bulk", chunk, 4096, "GB/s"))
        plan.append(("store_warp", chunk, 4096, "GB/s"))
    for lg in (12, 16, 20, 24):
        plan.append(("l2_red", lg, 0, "G rows/s"))
    for name, p, p2, unit in plan:
        try:
            v = eiger.probe(name, p, p2)
            print(json.dumps({"probe": name, "param": p, "param2": p2, "value": round(v, 2), "unit": unit}), flush=True)
        except eiger.EigerError as e:
            print(json.dumps({"probe": name, "param": p, "param2": p2, "error": str(e)}), flush=True)
    eiger.probe("release")


if __name__ == "__main__":
    main()
