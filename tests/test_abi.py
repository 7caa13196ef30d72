"""The C-ABI library loads and exports every symbol include/gm.h declares; argument
validation returns the documented codes.  No compute call needs a GPU here."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2404_07780_b200 import build as gm_build
    return C.CDLL(str(gm_build.build()))


def declared_symbols():
    text = (ROOT / "include" / "gm.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gm_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert {"gm_render", "gm_loss_grad", "gm_fit", "gm_workspace_bytes", "gm_strerror", "gm_version",
            "gm_render_host", "gm_loss_grad_host", "gm_fit_host"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_version_and_strerror(lib):
    lib.gm_version.restype = C.c_int
    lib.gm_strerror.restype = C.c_char_p
    assert lib.gm_version() >= 101
    assert b"invalid" in lib.gm_strerror(-1) and b"ok" == lib.gm_strerror(0)


def test_validation_codes_without_gpu():
    import numpy as np
    import paper_2404_07780_b200 as gm
    from paper_2404_07780_b200 import binding as bd
    from gen import models
    model = models.single_sersic()
    assert gm.gm_workspace_bytes(model, 16, 64, 64, 15) > 16 * 64 * 64 * 4
    assert gm.gm_workspace_bytes(model, 16, 64, 64, 14) == 0        # even K
    assert gm.gm_workspace_bytes(model, 16, 64, 64, 43) == 0        # K over GM_MAX_K
    assert gm.gm_workspace_bytes(model, 0, 64, 64, 15) == 0
    bad = {"n_par": 7, "components": [{"kind": "sersic", "convolve": 1, "slots": {"amp": 2, "s0": 9}}]}
    assert gm.gm_workspace_bytes(bad, 4, 32, 32, 5) == 0           # slot index out of range
    # null pointers are rejected before anything is launched (no GPU needed)
    m = bd._model_struct(model)
    b = bd._Batch(4, 32, 32, 5, None, None, None, None, 0)
    L = bd._lib()
    assert L.gm_render(C.byref(m), C.byref(b), None, None, None, 0, None) == -1
    assert L.gm_fit(C.byref(m), C.byref(b), None, None, None, None, None, None, 0, None) == -1


def test_options_and_init_entry_points(lib):
    # gm_set_option / gm_get_option replace the environment-variable hooks of round 1
    lib.gm_set_option.restype = C.c_int; lib.gm_get_option.restype = C.c_int
    for opt in (0, 1, 2):
        assert lib.gm_get_option(opt) == 1
        assert lib.gm_set_option(opt, 0) == 0 and lib.gm_get_option(opt) == 0
        assert lib.gm_set_option(opt, 7) == 0 and lib.gm_get_option(opt) == 1
    assert lib.gm_set_option(99, 1) == -1 and lib.gm_get_option(-1) == -1
    assert lib.gm_measure_fp32_peak(0, None, None) == -1            # validated before any CUDA call
    text = (ROOT / "paper_2404_07780_b200" / "csrc" / "gm_api.cu").read_text()
    assert "getenv" not in text and "cudaMemcpyToSymbol(" not in text


def test_binding_checks_shapes_before_the_library_sees_them():
    import torch
    from paper_2404_07780_b200 import binding as bd
    z = torch.zeros
    with pytest.raises(ValueError):
        bd._batch_struct(4, 16, 16, z(3, 5, 5), host=False)          # per-galaxy PSFs: 3 for 4 galaxies
    with pytest.raises(ValueError):
        bd._batch_struct(4, 16, 16, z(5, 7), host=False)             # not square
    with pytest.raises(ValueError):
        bd._batch_struct(4, 16, 16, z(5, 5), data=z(4, 16, 15), host=False)


def test_binding_refuses_cpu_tensors():
    import torch
    import paper_2404_07780_b200 as gm
    from gen import models
    with pytest.raises(TypeError):
        gm.gm_render(models.single_sersic(), torch.zeros(2, 7), 16, 16, torch.zeros(5, 5))


def test_loglike_eq17_host_helper():
    """gm_loglike (Eq. 17; k of P:204) against scipy's chi^2 log-density: a host helper, no GPU."""
    import numpy as np
    from scipy import stats
    import paper_2404_07780_b200 as gm
    chi2 = np.array([3.5, 16000.0, 14321.7, 1e-3, 0.0, np.inf, 50.0], dtype=np.float32)
    n_used = np.array([12, 16384, 14746, 9, 100, 100, 7], dtype=np.int32)
    out = gm.gm_loglike(chi2, n_used, 7)
    k = n_used.astype(np.float64) - 7
    for b in range(4):
        # ln Gamma(k/2) ~ 6e4 at k = 16377: fp64 rounding of the cancelling terms is ~1e-11 absolute
        assert out[b] == pytest.approx(stats.chi2.logpdf(float(chi2[b]), k[b]), rel=1e-12, abs=1e-9)
    assert np.isnan(out[4]) and np.isnan(out[5]) and np.isnan(out[6])      # chi2 = 0, inf, k = 0
    # the mode of the chi^2 density is k - 2: ln L falls off on either side of it
    m = gm.gm_loglike(np.array([98.0, 90.0, 106.0], dtype=np.float32), np.array([107] * 3, dtype=np.int32), 7)
    assert m[0] > m[1] and m[0] > m[2]
    with pytest.raises(gm.GmError):
        gm.gm_loglike(chi2, n_used, -1)
