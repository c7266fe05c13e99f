"""The oracle at other block sizes (block-size sweep; "block size ...
governs how many independent parsers the format exposes"; PAPER.md:102 sweeps 16 KB -> 4 KB).

`block_log2` is a header field of FORMAT.md section 1; the oracle is compiled for one value (`-DORA_BLOG`, 14 unless
ACEAPEX_BLOCK_LOG2 says otherwise). This file re-runs the pins that do not hard-wire 16 KiB against the 4 KiB and
32 KiB variants, each in its own interpreter: the hand-made containers of the independent Python writer (expected
bytes from the plain-definition `expand()`), round trips on adversarial sizes around the block size and on the five
profiles under both policies, the closed form for N equal bytes, decoder #1 == decoder #2 on every block, the
validator's promise checks, overlap / frequency-sum rejection, RAW streams by construction."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PINS = ("handmade_container or round_trip_adversarial or closed_form or zero_match or profiles_round_trip or "
        "thread_count or three_phase or overlapping or frequency_sum or validator_flags or raw_streams_decode or "
        "seek_aware")


@pytest.mark.parametrize("blog", [12, 15])
def test_oracle_pins_hold_at_other_block_sizes(blog):
    env = dict(os.environ, ACEAPEX_BLOCK_LOG2=str(blog))
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_codec.py"), "-q", "-x",
                        "-k", PINS, "-p", "no:cacheprovider"], env=env, cwd=ROOT, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-2000:]
    assert " passed" in r.stdout and "failed" not in r.stdout


def test_variant_refuses_a_container_of_another_block_size():
    """A 16 KiB container is E_FORMAT for the 4 KiB oracle and the other way round (header byte 12)."""
    code = ("import oracle, numpy as np\n"
            "c = oracle.encode(b'abcabcabcabc' * 500)\n"
            "assert c[12] == oracle.BLOG\n"
            "np.save('/tmp/aceapex_bs_%d.npy' % oracle.BLOG, c)\n")
    for blog in (12, 14):
        subprocess.run([sys.executable, "-c", code], env=dict(os.environ, ACEAPEX_BLOCK_LOG2=str(blog)), cwd=ROOT, check=True)
    check = ("import oracle, numpy as np\n"
             "c = np.load('/tmp/aceapex_bs_%d.npy' % (26 - oracle.BLOG))\n"
             "try:\n    oracle.decode_all(c)\nexcept oracle.OracleError as e:\n    assert e.code == -2, e.code\nelse:\n    raise SystemExit('accepted')\n")
    for blog in (12, 14):
        subprocess.run([sys.executable, "-c", check], env=dict(os.environ, ACEAPEX_BLOCK_LOG2=str(blog)), cwd=ROOT, check=True)
