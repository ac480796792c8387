"""`-m gpu`: the bounds-checked debug build (csrc/pic_check.cuh, libpic_b200_check.so) on a tour
of every kernel and mode; zero index violations.  Stands in for compute-sanitizer memcheck,
which is closed on this GPU pool."""
import os
import re
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def test_no_index_violations_in_the_check_build():
    from paper_1111_5295_b200 import binding as B
    B.load()
    assert B.debug_bounds() == -1                       # this process runs the production build
    env = dict(os.environ, PIC_B200_CHECK="1")
    r = subprocess.run([sys.executable, os.path.join(HERE, "bounds_check_driver.py")], env=env,
                       capture_output=True, text=True, timeout=1500)
    print(r.stdout[-2000:], r.stderr[-2000:])
    assert r.returncode == 0
    m = re.search(r"BOUNDS_VIOLATIONS=(-?\d+)", r.stdout)
    assert m and int(m.group(1)) == 0, r.stdout[-500:]
    assert int(re.search(r"MOVES=(\d+)", r.stdout).group(1)) > 400
