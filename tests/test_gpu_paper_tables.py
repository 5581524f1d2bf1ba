"""The paper's own accuracy experiment on the CUDA path (second half): Tables 1 and 2
(PAPER.md L128-L137, L158-L165), self-gravitating sheet, water-bag x0 = 1, p0 = 0.5 with its edges, x, p in [-2, 2],
periodic in both directions (L113, L145-L150), dt = 0.01 and 0.1, n = 256 ... 2048, eq (16) spline ("FD") and global
spline ("GS"): maximum relative error of the energy and of the norm over the run.

The run length is not stated in the paper (reading D13); t = 100 is used (P20: at dt = 0.1, n = 256 it reproduces
the printed 5e-4).  What is asserted, and why not more:
  * Table 2 (dt = 0.1), FD and GS, every n: the energy error within a factor 2.5 of the printed value;
  * Table 1 (dt = 0.01), n = 1024 and 2048: within a factor 3 (FD 3.8e-6 / 4.9e-6 against 1e-5 / 4e-6);
  * Table 1, n = 256 and 512: BELOW the printed values (6.5e-5 / 1.0e-5 against 7e-3 / 7e-4): the paper's coarse runs
    also lose 1e-3 / 1e-4 of the norm, which a constant shift per line cannot do on a periodic axis (reading D14) --
    here the norm is kept to round-off for every n, dt and spline, and the energy error with it.
The state of each run is also compared with the oracle where the oracle is fast enough (n = 256, dt = 0.1)."""
from __future__ import annotations

import os

import numpy as np
import pytest

from oracle import BC_PERIODIC, MODEL_SHEET, SPLINE_GS, Oracle
from paper_1206_3229_b200 import binding as vb
from paper_1206_3229_b200 import inputs

pytestmark = pytest.mark.gpu
DOM = (-2.0, 2.0, -2.0, 2.0)


def read_table(golden_dir, name):
    rows = {}
    for line in open(os.path.join(golden_dir, name)):
        if line.strip() and not line.startswith("#"):
            v = line.split()
            rows[int(v[0])] = [float(x) for x in v[1:]]
    return rows


def waterbag(n):
    x, p = inputs.nodes(DOM[0], DOM[1], n), inputs.nodes(DOM[2], DOM[3], n)
    return np.where((np.abs(x)[None, :] <= 1.0) & (np.abs(p)[:, None] <= 0.5), 0.5, 0.0)


def run(n, dt, gs, t_end=100.0):
    g = vb.Vlasov(MODEL_SHEET, (n, n), DOM, dt, bc_x=BC_PERIODIC, bc_p=BC_PERIODIC, **({"spline": vb.SPLINE_GS} if gs else {}))
    g.upload(waterbag(n))
    m0 = g.moments()
    de = dn = 0.0
    k = int(round(1.0 / dt))
    for _ in range(int(round(t_end))):
        g.step(k)
        m = g.moments()
        de = max(de, abs(m[7] - m0[7]) / abs(m0[7]))
        dn = max(dn, abs(m[1] - m0[1]) / m0[1])
    f = g.download()
    g.close()
    return de, dn, f


@pytest.mark.parametrize("gs", [0, 1], ids=["FD", "GS"])
@pytest.mark.parametrize("n", [256, 512, 1024, 2048])
def test_table2_dt_0p1(n, gs, golden_dir):
    paper = read_table(golden_dir, "sheet_table2_gs_L158.txt" if gs else "sheet_table2_L158.txt")[n][0]
    de, dn, _ = run(n, 0.1, gs)
    assert paper / 2.5 <= de <= paper * 2.5, (de, paper)
    assert dn <= 1e-12


@pytest.mark.parametrize("gs", [0, 1], ids=["FD", "GS"])
@pytest.mark.parametrize("n", [256, 512, 1024, 2048])
def test_table1_dt_0p01(n, gs, golden_dir):
    row = read_table(golden_dir, "sheet_table1_L128.txt")[n]
    paper = row[2] if gs else row[0]
    de, dn, _ = run(n, 0.01, gs)
    if n >= 1024:
        assert paper / 3.0 <= de <= paper * 3.0, (de, paper)
    else:
        assert de <= paper, (de, paper)   # the paper's coarse runs lose norm (D14); this path does not
    assert dn <= 1e-12


@pytest.mark.parametrize("gs", [0, 1], ids=["FD", "GS"])
def test_the_tables_run_matches_the_oracle(gs):
    n = 256
    _, _, f = run(n, 0.1, gs, t_end=20.0)
    o = Oracle(MODEL_SHEET, (n, n), DOM, 0.1, threads=os.cpu_count() or 8, bc_x=BC_PERIODIC, bc_p=BC_PERIODIC,
               **({"spline": SPLINE_GS} if gs else {}))
    o.upload(waterbag(n))
    o.step(200)
    assert np.max(np.abs(f - o.download())) <= 1e-10 * np.max(np.abs(f))
    o.close()
