"""Race / bounds evidence without the sanitizer (-m gpu): the -DTWK_DEBUG build of the same sources counts violations of
the kernels' own invariants (record ids inside the arena, angles sorted after every merge, the sorted list a permutation
of the ids, one writer per record per re-judging phase, worklist slots in range, new angles inside their intervals).
Run on the inputs that drive the data-dependent paths hardest: the Fig.1 / Fig.2 sources, the caustic band of config 4,
low-q lenses, with the slope detector's gate opened so that the re-judging rounds run."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import json, sys
import numpy as np
sys.path.insert(0, %r)
import paper_2501_03322_b200 as P
import workloads as W
assert "TWK_DEBUG" in P.twk_version(), P.twk_version()
full = W.config4()
zc = full.zeta[:, 0] + 1j * full.zeta[:, 1]
band = np.where((np.abs(zc.imag) < 0.25) & (np.abs(zc.real) < 0.6))[0]
cases = [W.fig2_case(), W.fig1_case(), full.subset(band[:: max(1, len(band) // 3000)]), W.lowq_sweep(n=1500),
         W.config2().subset(np.arange(4800, 5200))]
P.twk_debug_counters(reset=True)
res = {}
for gate, cs in ((1e-5, 0.70710678118654752), (1e30, 0.2), (1e30, 0.0)):
    for slots in (-1, 0):
        c = P.Context(4096, slope_gate=gate, slope_cos=cs, handoff_slots=slots)
        for wl in cases:
            for tol in (1e-4, 1e-6, 1e-12):
                if tol == 1e-12 and wl.n_sources > 4:
                    continue
                r = c.magnify_workload(wl, tol)
                assert np.all(np.isfinite(r["mu"]))
        c.close()
print(json.dumps(P.twk_debug_counters()))
"""


def test_debug_build_invariants_hold():
    from paper_2501_03322_b200 import build
    lib = build.build(debug=True)
    env = dict(os.environ, TWK_LIBRARY=lib)
    out = subprocess.run([sys.executable, "-c", CHILD % ROOT], env=env, capture_output=True, text=True, timeout=1500)
    assert out.returncode == 0, out.stderr[-3000:]
    c = json.loads(out.stdout.strip().splitlines()[-1])
    assert c[:6] == [0, 0, 0, 0, 0, 0], c          # no violation of any invariant
    assert c[6] > 10000 and c[7] > 20000, c         # ... and the checks ran: sources and iterations checked
    # stage 1.5 took part: entries taken up >= entries solved >= sources finished there > 0; some were passed on unread
    # (the handoff_slots = 0 contexts do not launch it)
    assert c[8] >= c[9] >= c[10] > 1000 and c[11] > 0, c


def test_release_build_has_no_debug_counters():
    import paper_2501_03322_b200 as P
    assert "TWK_DEBUG" not in P.twk_version()
    with pytest.raises(P.TwkError):
        P.twk_debug_counters()
