"""GPU parity of the opt-in kernel variants (selected once per process by environment switches, hence subprocesses):
TDDFT_VAR bit 6 = TMA-staged inverse plane kernel (72 x 72 planes only), TDDFT_CT_FULL=0 = row-block contraction kernels,
TDDFT_VAR=0 = non-persistent plane grids without prefetch / eviction hints.  Same tolerance as the default path."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import sys
sys.path.insert(0, %(root)r); sys.path.insert(0, %(root)r + "/tests")
from helpers import Case, rel_fro
case = Case.from_config(3, nocc=(5, 4), fft_backend="numpy", pair_tile=3)
for mode in (0, 1):
    X = case.trial(2, mode)
    err = rel_fro(case.gpu_apply(X, mode), case.oracle.apply(X, mode))
    assert err < 1e-10, (mode, err)
print("variant ok")
"""


@pytest.mark.parametrize("env", [{"TDDFT_VAR": "113"}, {"TDDFT_CT_FULL": "0"}, {"TDDFT_VAR": "0"}])
def test_variant_parity_on_the_bench_grid(env):
    e = dict(os.environ); e.update(env)
    r = subprocess.run([sys.executable, "-c", SCRIPT % {"root": ROOT}], env=e, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "variant ok" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]
