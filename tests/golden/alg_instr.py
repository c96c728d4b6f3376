"""Writes tests/golden/alg_instr_per_pair.json: the ALGORITHMIC thread-instructions per annihilation pair of the transport
kernel for each bench workload = the oracle's event counts per pair x the least instruction cost of each event (the
audit table of DESIGN.md section 6; SURVEY.md 8(d) arrives at 740 for C1 by the same method).  Calls only oracle/.

    python tests/golden/alg_instr.py            # ~1 minute; rewrites the json next to this file
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

# least thread-instructions per event: a Philox block is 56; FMA = 1
COST = dict(source=124, voxel_pick=140, search_ring=89, search_list=346, entry=35, step=75, exit=25, lookup=68, outcome=19, hit=20,
            kn_trial=80, compton_accept=46, rayleigh=60, phantom_step=95, phantom_outcome=19)


def per_pair(c, n, ring, voxel):
    ev = dict(source=n, voxel_pick=n if voxel else 0, entry=c["entries"], step=c["steps"], exit=c["exits"],
              lookup=c["steps"] - c["exits"], outcome=c["steps"] - c["exits"] - c["step_vacuum"], hit=c["hits"],
              kn_trial=c["kn_trials"], compton_accept=c["compton"] + c["ph_compton"], rayleigh=c["rayleigh"],
              phantom_step=c["ph_steps"], phantom_outcome=c["ph_compton"] + c["ph_absorbed"])
    ev["search_ring" if ring else "search_list"] = c["searches"]
    return sum(COST[k] * v for k, v in ev.items()) / n, {k: v / n for k, v in ev.items()}


def main():
    from oracle import gpet_oracle as O
    from paper_2603_07327_b200 import workloads as W
    T = W.tables()
    out = {}
    for cfg, idx, n in (("C1", 0, 2_000_000), ("C2", 0, 2_000_000), ("C3", 0, 2_000_000), ("C3", 10, 2_000_000), ("C4", 0, 2_000_000),
                        ("P1", 0, 2_000_000), ("T1", 0, None), ("T2", 0, None), ("T3", 0, None)):
        r = W.config_runs(cfg, n)[idx]
        res = O.simulate(r.geometry, T, r.source, r.n_pairs, r.seed, threads=os.cpu_count() or 1)
        total, ev = per_pair(res.counters, r.n_pairs, ring=r.geometry.panel_pose is None, voxel=r.source.kind == 1)
        out[r.name] = dict(instr_per_pair=round(total, 1), events_per_pair={k: round(v, 4) for k, v in ev.items()}, pairs=r.n_pairs)
        print(r.name, round(total, 1))
    out["_cost_per_event"] = COST
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "alg_instr_per_pair.json"), "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
