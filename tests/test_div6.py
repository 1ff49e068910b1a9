"""Host-side check of the quotient the fp32 convdiff kernel forms without a division (csrc/wl_convdiff.cuh, cd_div6): the
multiply-and-correct sequence equals IEEE x / 6 for every finite |x| >= 2^-100.  Scaling by a power of two is exact, so all
2^23 mantissas of one binade, both signs, cover the normal range; the binades at both ends of the guarded range and the largest
binade are swept as well (tests/div6_check.c, compiled here with gcc; IEEE arithmetic is the same on host and device)."""
import os
import struct
import subprocess
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))


def _bits(x: float) -> int:
    return struct.unpack("<I", struct.pack("<f", x))[0]


def test_multiply_and_correct_quotient_is_the_ieee_quotient():
    with tempfile.TemporaryDirectory() as d:
        exe = os.path.join(d, "div6_check")
        subprocess.run(["gcc", "-O2", "-mfma", "-ffp-contract=off", os.path.join(HERE, "div6_check.c"), "-o", exe, "-lm"], check=True)
        spans = []
        for lo in (1.0, 2.0 ** -100, 2.0 ** -99, 2.0 ** 126, 2.0 ** 127):     # whole binades [lo, 2 lo)
            spans.append((_bits(lo), 1 << 23))
            spans.append((_bits(-lo), 1 << 23))
        for first, count in spans:
            out = subprocess.run([exe, str(first), str(count)], check=True, capture_output=True, text=True).stdout
            assert int(out) == 0, (hex(first), out)
