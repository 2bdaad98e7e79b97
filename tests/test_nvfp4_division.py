"""The division step of the NVFP4 quantisers (paper_2606_19004_b200/csrc/nvfp4_math.cuh, BlockDivisor), restated in C
and checked EXHAUSTIVELY against the host's IEEE division: for each of the eight significands (1 + k/8) an E4M3 scale
can have, and all 2^23 significands of the dividend,
    q = RN(x * y);  r = fma(-sf, q, x);  q' = fma(r, y, q)      with y = RN(1 / sf)
equals RN(x / sf) bit for bit (reading N3: the quotient that decides an E2M1 code is the fp32
IEEE quotient on both sides).  Powers of two scale dividend, divisor and quotient exactly, so the significands are all
that matters; 6 = 1.5 * 4 (the block maximum / 6) is one of the eight.  Dropping the correction step fails the check.
"""
import os
import shutil
import subprocess
import tempfile

import pytest

SRC = r"""
#include <math.h>
#include <stdio.h>
#include <stdint.h>
#include <string.h>
static inline float div_seq(float x, float sf, float y) {
  float q = x * y;
#ifndef NO_CORRECTION
  float r = fmaf(-sf, q, x);
  q = fmaf(r, y, q);
#endif
  return q;
}
int main(void) {
  long bad = 0, n = 0;
  for (int k = 0; k < 8; ++k) {
    volatile float sf = 1.0f + k / 8.0f, one = 1.0f;
    const float y = one / sf;                       /* RN(1 / sf): what __frcp_rn returns */
    for (uint32_t m = 0; m < (1u << 23); ++m) {
      const uint32_t bits = 0x3f800000u | m;
      float x;
      memcpy(&x, &bits, 4);
      volatile float xv = x;
      const float ref = xv / sf, got = div_seq(x, sf, y);
      bad += memcmp(&ref, &got, 4) != 0;
      ++n;
    }
  }
  printf("%ld %ld\n", n, bad);
  return 0;
}
"""


def _run(flags):
    with tempfile.TemporaryDirectory() as d:
        c, exe = os.path.join(d, "div.c"), os.path.join(d, "div")
        with open(c, "w") as f:
            f.write(SRC)
        subprocess.run(["gcc", "-O2", "-ffp-contract=off", *flags, c, "-o", exe, "-lm"], check=True)
        n, bad = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
        return int(n), int(bad)


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_block_divisor_sequence_is_ieee_division_for_every_significand():
    n, bad = _run([])
    assert n == 8 << 23 and bad == 0


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_the_check_sees_a_missing_correction_step():
    n, bad = _run(["-DNO_CORRECTION"])
    assert bad > 1000
