"""-m gpu: the nu_n table set-up against CUDA stream capture (include/gm.h, "Process-wide state").

The table is filled by a kernel on the stream of the first call and later calls wait for it through an
event recorded there; neither belongs inside a captured graph.  So a compute call (or gm_init) on a
CAPTURING stream while the table is missing is refused with GM_EINVAL and enqueues nothing, and gm_init
returns only after the table is complete.  Needs a process in which libgm has not run yet, hence the
subprocess."""
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent

CODE = r"""
import torch
import paper_2404_07780_b200 as gm
from gen import models
model = models.single_sersic()
par = torch.tensor([[32.3, 31.1, 1.0, 6.0, 2.0, 0.7, 0.4]] * 3, device="cuda")
psf = torch.zeros(5, 5, device="cuda"); psf[2, 2] = 1.0
out = torch.zeros(3, 64, 64, device="cuda")
ws = torch.empty(gm.gm_workspace_bytes(model, 3, 64, 64, 5) + 256, dtype=torch.uint8, device="cuda")
torch.cuda.synchronize()
side = torch.cuda.Stream()
g = torch.cuda.CUDAGraph()
refused = []
try:
    with torch.cuda.graph(g, stream=side):
        for call in (lambda: gm.gm_init(), lambda: gm.gm_render(model, par, 64, 64, psf, out=out, workspace=ws)):
            try:
                call()
            except gm.GmError as e:
                refused.append(e.status)
except Exception as e:                       # an empty capture may itself complain; not what is tested
    print("capture exit:", type(e).__name__)
assert refused == [-1, -1], refused
assert gm.gm_last_launch_count() == 0
torch.cuda.synchronize()
assert float(out.abs().sum()) == 0.0         # nothing ran
gm.gm_init()                                 # outside a capture: builds the table and waits for it
gm.gm_init()                                 # idempotent
img = gm.gm_render(model, par, 64, 64, psf, out=out, workspace=ws)
torch.cuda.synchronize()
assert float(img.sum()) > 0.0 and bool(torch.isfinite(img).all())
print("INIT_CAPTURE_OK")
"""


def test_table_setup_is_refused_inside_a_capture_and_gm_init_completes_it():
    r = subprocess.run([sys.executable, "-c", CODE], cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "INIT_CAPTURE_OK" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
