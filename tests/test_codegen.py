"""The committed generated header is reproducible from the committed generator: regenerating
`csrc/mms_generated.cuh` under a DIFFERENT hash seed gives the tracked file byte for byte.  CPU only (SymPy)."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TRACKED = os.path.join(ROOT, "paper_2607_05668_b200", "csrc", "mms_generated.cuh")


def test_generated_header_is_reproducible(tmp_path):
    out = str(tmp_path / "mms_generated.cuh")
    env = dict(os.environ, PYTHONHASHSEED="20261105", PYTHONPATH=ROOT)      # any seed: nothing may depend on set / hash order
    r = subprocess.run([sys.executable, "-m", "paper_2607_05668_b200.gen.mms_codegen", out], cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stderr[-2000:]
    with open(out, "rb") as a, open(TRACKED, "rb") as b:
        new, old = a.read(), b.read()
    assert new == old, ("csrc/mms_generated.cuh differs from what gen/mms_codegen.py emits "
                        f"({len(new)} vs {len(old)} bytes): regenerate it with `python -m paper_2607_05668_b200.gen.mms_codegen`")
