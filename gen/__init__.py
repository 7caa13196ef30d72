"""Seeded synthetic input generators shared by tests, bench and smoke.

Holds NONE of the method's arithmetic: model descriptions are plain data,
PSFs are analytic input images, noise is drawn around a truth image that the
caller renders (oracle in tests, CUDA path in bench).
"""
from . import configs, models, psf  # noqa: F401
