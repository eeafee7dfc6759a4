"""Sampled rows that a GPU run saved (THC_ROWS_SAVE=<file> with tests/test_gpu_rows.py) against the stored oracle rows of
tests/golden/ -- for terms whose oracle row was not there yet when the GPU ran (a config-4 sigma6 row takes hours of CPU).
Opt-in: THC_GPU_ROWS_FILE=<file.npz>.  Same tolerance as the online test: 1e-10 of the term's largest element in the row."""
import os

import numpy as np
import pytest

from golden.make_rows import load_rows


@pytest.mark.skipif(not os.environ.get("THC_GPU_ROWS_FILE"), reason="set THC_GPU_ROWS_FILE to an .npz written with THC_ROWS_SAVE")
def test_saved_gpu_rows_match_the_stored_oracle_rows():
    data = np.load(os.environ["THC_GPU_ROWS_FILE"])
    cfg, rows = int(data["cfg"]), [int(p) for p in data["rows"]]
    gdir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    errs = {}
    for n, P in enumerate(rows):
        for term, want in load_rows(gdir, cfg, P).items():
            errs[(P, term)] = np.abs(data[term][n] - want).max() / np.abs(want).max()
    assert errs, "no stored oracle row for the saved rows"
    print(f"config {cfg} saved GPU rows vs stored oracle rows: { {f'{t}@{P}': float(e) for (P, t), e in errs.items()} }")
    assert all(e <= 1e-10 for e in errs.values()), errs
