"""Writes tests/golden/tiny_oracle_expected.txt: the oracle's results on BASELINE.json configs[0] ("tiny").

    python tests/golden/make_golden.py

Calls ONLY oracle/ (and the shared seeded input generator, which holds no method arithmetic).  The stored values
guard the oracle against silent changes (a later edit of its arithmetic must regenerate this file and say why in
the commit message); they are never produced by the CUDA path.
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle  # noqa: E402
from paper_2606_10537_b200 import workloads as W  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle_expected.txt")


def compute():
    w = W.CONFIGS["tiny"]
    inp = W.make_inputs(w, threads=1)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    sha = hashlib.sha256()
    for k in ("Q_dec", "Kcache", "Vcache", "K_dec", "V_dec", "keep"):
        sha.update(np.ascontiguousarray(inp[k]).tobytes())
    lines = ["# oracle.step on workloads.CONFIGS['tiny'] (BASELINE.json configs[0]); written by tests/golden/make_golden.py",
             f"inputs_sha256 = {sha.hexdigest()}"]
    lines.append("chunk_ids = " + " ".join(str(int(x)) for x in ref["ids"].ravel()))
    lines.append("scores = " + " ".join(f"{x:.12e}" for x in ref["scores"].ravel()))
    lines.append("gather_idx_head0 = " + " ".join(str(int(x)) for x in ref["gather_idx"][0, 0]))
    lines.append("LSE_row0_per_head = " + " ".join(f"{x:.12e}" for x in ref["LSE"][0, :, 0]))
    lines.append("O_head0_row0_first8 = " + " ".join(f"{x:.12e}" for x in ref["O"][0, 0, 0, :8]))
    lines.append(f"O_abs_sum = {np.abs(ref['O']).sum():.12e}")
    lines.append(f"LSE_sum = {ref['LSE'].sum():.12e}")
    return "\n".join(lines) + "\n"


if __name__ == "__main__":
    with open(OUT, "w") as f:
        f.write(compute())
    print("wrote", OUT)
