"""Fixtures under tests/golden/ (values the paper prints) against the input module and the
bookkeeping formulas Eqs. (8)-(10)."""
import os

import fh_inputs as fi

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _table_s2():
    rows = []
    for line in open(os.path.join(GOLD, "table_s2.txt")):
        line = line.strip()
        if line and not line.startswith("#"):
            n, tj, d = (int(x) for x in line.split())
            rows.append((n, tj, d))
    return rows


def test_table_s2_caption_totals():
    rows = _table_s2()
    assert len(rows) == 32                                        # "32 sectors" (caption)
    assert sum(d for _, _, d in rows) == 12288                    # chi_SU(2), Eq. (10)
    chi = sum(d * (tj + 1) for _, tj, d in rows)                  # Eq. (8)
    assert chi == 30842 and abs(chi - 30000) / 30000 < 0.03       # "chi ~ 30000"
    assert max(d for _, _, d in rows) == 1735                     # d_max, Eq. (9)
    assert all((n + tj) % 2 == 0 for n, tj, _ in rows)            # parity rule n + 2j even
    assert 2.4 <= chi / 12288 <= 2.6                              # "chi ~ 2.4 chi_SU(2)" PAPER.md:47, 233


def test_input_module_table_s2_equals_fixture():
    gold = {(n, tj): d for n, tj, d in _table_s2()}
    assert fi.table_s2_profile() == gold
