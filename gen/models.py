"""Model descriptions as plain data (no arithmetic of the method lives here).

A model is ``{"n_par": P, "names": [...], "roles": [...], "components": [...]}``.
Each component is ``{"kind": str, "convolve": 0|1, "slots": {slot: index}}``
with slot names ``xc yc theta q amp s0 s1 s2 box m0`` (paper: P:35 p = {p_G, p_L};
P:61 summed components; P:322-327 shared parameters; P:598 psf flag).  ``box`` is the
boxiness B of Eq. 2.  A used ``m0`` slot (the zero point) means the
``amp`` slot holds a magnitude m and the intensity follows Eq. 5 / 8 / 10 / 15.

    Sersic   amp=Ie  s0=re    s1=n           (Eq. 1)
    ExpDisk  amp=I0  s0=rs                   (Eq. 7)
    Ferrer   amp=I0  s0=r_out s1=a  s2=b     (Eq. 9)
    King     amp=I0  s0=rc    s1=rt s2=alpha (Eq. 11)
    Gaussian amp=I0  s0=FWHM                 (Eq. 12)
    Moffat   amp=I0  s0=FWHM  s1=n           (Eq. 13)
    Sky      amp=I_sky                       (Eq. 16)

``roles`` drive the default fit options (step size, bounds, log10 space) of
``gen.configs.fit_options``: one of
``cx cy amp radius index q theta shape sky box mag zeropoint``.
"""
from __future__ import annotations


def _model(names, roles, components):
    assert len(names) == len(roles)
    return {"n_par": len(names), "names": list(names), "roles": list(roles),
            "components": components}


def single_sersic():
    """BASELINE configs C0-C2: P = 7, [xc, yc, Ie, re, n, q, theta]."""
    return _model(
        ["xc", "yc", "Ie", "re", "n", "q", "theta"],
        ["cx", "cy", "amp", "radius", "index", "q", "theta"],
        [{"kind": "sersic", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}}])


def bulge_disk():
    """BASELINE config C3: Sersic bulge + exponential disk, shared centre, P = 11."""
    return _model(
        ["xc", "yc", "b_Ie", "b_re", "b_n", "b_q", "b_theta", "d_I0", "d_rs", "d_q", "d_theta"],
        ["cx", "cy", "amp", "radius", "index", "q", "theta", "amp", "radius", "q", "theta"],
        [{"kind": "sersic", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}},
         {"kind": "expdisk", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 7, "s0": 8, "q": 9, "theta": 10}}])


def sersic_bar_nucleus():
    """BASELINE config C4: Sersic + Ferrer bar + circular Moffat nucleus, shared
    centre, P = 2 + 5 + 6 + 3 = 16 (the nucleus carries no q/theta)."""
    return _model(
        ["xc", "yc", "s_Ie", "s_re", "s_n", "s_q", "s_theta",
         "f_I0", "f_rout", "f_a", "f_b", "f_q", "f_theta", "m_I0", "m_fwhm", "m_n"],
        ["cx", "cy", "amp", "radius", "index", "q", "theta",
         "amp", "radius", "shape", "shape", "q", "theta", "amp", "radius", "shape"],
        [{"kind": "sersic", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}},
         {"kind": "ferrer", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 7, "s0": 8, "s1": 9, "s2": 10, "q": 11, "theta": 12}},
         {"kind": "moffat", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 13, "s0": 14, "s1": 15}}])


def all_profiles():
    """Parity-only model: every built-in profile once (Sec. 4.1-4.2.6), with an
    unconvolved Gaussian point source and a flat sky (Eq. 16).
    Centre shared by the first four, P = 30."""
    names = ["xc", "yc",
             "se_Ie", "se_re", "se_n", "se_q", "se_th",
             "ex_I0", "ex_rs", "ex_q", "ex_th",
             "fe_I0", "fe_rout", "fe_a", "fe_b", "fe_q", "fe_th",
             "ki_I0", "ki_rc", "ki_rt", "ki_al", "ki_q", "ki_th",
             "ga_x", "ga_y", "ga_I0", "ga_fwhm",
             "mo_I0", "mo_fwhm",
             "sky"]
    roles = ["cx", "cy",
             "amp", "radius", "index", "q", "theta",
             "amp", "radius", "q", "theta",
             "amp", "radius", "shape", "shape", "q", "theta",
             "amp", "radius", "radius", "shape", "q", "theta",
             "cx", "cy", "amp", "radius",
             "amp", "radius",
             "sky"]
    comps = [
        {"kind": "sersic", "convolve": 1,
         "slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}},
        {"kind": "expdisk", "convolve": 1,
         "slots": {"xc": 0, "yc": 1, "amp": 7, "s0": 8, "q": 9, "theta": 10}},
        {"kind": "ferrer", "convolve": 1,
         "slots": {"xc": 0, "yc": 1, "amp": 11, "s0": 12, "s1": 13, "s2": 14, "q": 15, "theta": 16}},
        {"kind": "king", "convolve": 1,
         "slots": {"xc": 0, "yc": 1, "amp": 17, "s0": 18, "s1": 19, "s2": 20, "q": 21, "theta": 22}},
        {"kind": "gaussian", "convolve": 0,
         "slots": {"xc": 23, "yc": 24, "amp": 25, "s0": 26}},
        # Moffat with a FIXED concentration index is not expressible (every slot
        # is a parameter), so the test model ties its index to the Sersic n slot.
        {"kind": "moffat", "convolve": 1,
         "slots": {"xc": 23, "yc": 24, "amp": 27, "s0": 28, "s1": 4}},
        {"kind": "sky", "convolve": 0, "slots": {"amp": 29}},
    ]
    return _model(names, roles, comps)


def one_component(kind: str, convolve: int = 1, box: bool = False, mag: bool = False):
    """Single component of the given kind with its own full geometry; ``box`` adds the
    boxiness B (Eq. 2), ``mag`` the magnitude parameterisation (amp slot = m, plus m0)."""
    shape = {"sersic": (["Ie", "re", "n"], ["amp", "radius", "index"]),
             "expdisk": (["I0", "rs"], ["amp", "radius"]),
             "ferrer": (["I0", "rout", "a", "b"], ["amp", "radius", "shape", "shape"]),
             "king": (["I0", "rc", "rt", "alpha"], ["amp", "radius", "radius", "shape"]),
             "gaussian": (["I0", "fwhm"], ["amp", "radius"]),
             "moffat": (["I0", "fwhm", "n"], ["amp", "radius", "shape"])}[kind]
    names = ["xc", "yc", "theta", "q"] + shape[0]
    roles = ["cx", "cy", "theta", "q"] + shape[1]
    slots = {"xc": 0, "yc": 1, "theta": 2, "q": 3, "amp": 4}
    for k in range(len(shape[0]) - 1):
        slots[f"s{k}"] = 5 + k
    if mag:
        names[4] = "mag"; roles[4] = "mag"
    if box:
        slots["box"] = len(names); names.append("box"); roles.append("box")
    if mag:
        slots["m0"] = len(names); names.append("m0"); roles.append("zeropoint")
    return _model(names, roles, [{"kind": kind, "convolve": convolve, "slots": slots}])


def boxy_bulge_disk_mag():
    """Parity model for SURVEY 8(f)-2: boxy Sersic bulge + disky exponential disk, both
    in magnitudes with one shared zero point, shared centre, P = 14."""
    return _model(
        ["xc", "yc", "b_mag", "b_re", "b_n", "b_q", "b_theta", "b_box",
         "d_mag", "d_rs", "d_q", "d_theta", "d_box", "m0"],
        ["cx", "cy", "mag", "radius", "index", "q", "theta", "box",
         "mag", "radius", "q", "theta", "box", "zeropoint"],
        [{"kind": "sersic", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6, "box": 7, "m0": 13}},
         {"kind": "expdisk", "convolve": 1,
          "slots": {"xc": 0, "yc": 1, "amp": 8, "s0": 9, "q": 10, "theta": 11, "box": 12, "m0": 13}}])
