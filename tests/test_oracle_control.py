"""Control for reading R12: the oracle proper defines the packet state between steps in fp32 where
the 48-byte record and the queue store it (cell-local position, q, u, v).  Those two roundings entered the oracle
after the first kernel existed, so this file shows what they do and do not change, without any GPU:

  * every pin of tests/test_oracle_pins.py also holds on the control build with the roundings off
    (-DORA_STATE_FP32=0, pure fp64 state; tables, B^ and n^ stay fp32 as in the oracle's first commit);
  * on the five workloads the two builds produce image maps of the same packet ids that agree within 3 sigma
    per pixel and 0.5 % integrated, and the fraction of packets whose event sequences agree between the two
    builds is printed (it is < 1 only through the chaotic amplification of a last-bit difference, which is
    the reason the state is defined in fp32: both implementations then decide on identical numbers).
"""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2512_01283_b200 import inputs
from harness import oracle_run, compare_sequences, show

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SMALL = {
    "c1": dict(n=32, n_packets=20000, npix=64),
    "c2": dict(n=48, n_packets=6000, npix=64),
    "c3": dict(n=12, n_packets=1500, npix=32),
    "c4": dict(n=40, n_packets=4000, npix=48),
    "c5": dict(n=32, n_packets=3000, npix=48),
}


def test_pins_hold_on_the_pure_fp64_state_build():
    env = dict(os.environ, KRP_ORACLE_VARIANT="pure")
    p = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                        "-p", "no:cacheprovider"], env=env, capture_output=True, text=True, timeout=1200)
    assert p.returncode == 0, p.stdout[-3000:] + p.stderr[-2000:]
    assert " passed" in p.stdout and "failed" not in p.stdout


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4", "c5"])
def test_rounded_and_pure_oracle_images_agree(name):
    cfg = inputs.make(name, **SMALL[name])
    n = cfg["n_packets"]
    ev_r, img_r, img2_r, st_r = oracle_run(cfg, 0, n)
    ev_p, img_p, img2_p, st_p = oracle_run(cfg, 0, n, variant="pure")
    frac, info = compare_sequences(ev_p, ev_r, np.arange(n), pos_tol=2e-3)
    print("R12 control %s: rounded-state oracle vs pure-fp64 oracle, sequences agree for %.5f of %d packets %s"
          % (name, frac, n, show(info)))
    # the roundings change no statistic: same maps within the Monte-Carlo noise of the sample, per pixel and integrated
    I_o = img_p[:, 0].sum()
    for s in range(3):
        a, b = img_r[:, s].sum(), img_p[:, s].sum()
        assert abs(a - b) <= 0.005 * max(abs(b), 1e-3 * I_o), (name, s, a, b)
    # per pixel: the two maps differ only by the contributions of the packets that disagree, which sit in one map or the
    # other, so the noise of the difference is that of both samples
    sigma = np.sqrt(img2_p + img2_r)
    bad = np.abs(img_r - img_p) > 3 * sigma + 1e-9 * img_p[:, 0].max()
    assert bad.sum() == 0, (name, int(bad.sum()))
    for k in ("w_escaped", "w_absorbed", "w_cut"):
        assert abs(st_r[k] - st_p[k]) <= 3e-3 * n, (k, st_r[k], st_p[k])
    # a single fp32 rounding of (q,u,v) and of a cell-local coordinate cannot move most packets
    assert frac >= 0.95, show(info)
