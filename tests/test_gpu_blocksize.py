"""Block-size variants of the CUDA library (-DACEAPEX_BLOCK_LOG2, `bench.py --sweep`) against the
oracle variant of the same size, each in its own interpreter (a process loads one library)."""
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("blog", [12, 13, 15])
def test_block_size_variant_matches_the_oracle_variant(blog):
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; the product has no CPU fallback")
    sys.path.insert(0, ROOT)
    from paper_2606_24531_b200 import build as B_
    lib = B_.build_variant(f"block_log2{blog}", {"ACEAPEX_BLOCK_LOG2": blog})
    env = dict(os.environ, ACEAPEX_BLOCK_LOG2=str(blog), ACEAPEX_LIB=lib)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "blocksize_gpu_check.py")], env=env, cwd=ROOT,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "blocksize check ok" in r.stdout, r.stdout[-2000:] + r.stderr[-3000:]
