"""The C-ABI driven from a compiled C99 program (tests/c_abi_driver.c): cudaMalloc'ed arena,
layup_init, layup_round, layup_sync, layup_weights, layup_last_order, with no Python struct in
between.  K = 2 makes the expected result exact: both replicas end at the average and the
push-sum weights sum to 1."""
import subprocess

import pytest

from test_library_cpu import _cc

pytestmark = pytest.mark.gpu


def test_c_program_drives_the_library(tmp_path):
    from paper_2410_05985_b200.build import build
    build()
    r = subprocess.run([_cc(tmp_path, [], True)], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "C_ABI_OK" in r.stdout, (r.stdout, r.stderr)
