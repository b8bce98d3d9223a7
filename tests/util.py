"""Helpers shared by the tests (no method arithmetic)."""
import functools

import numpy as np

import oracle
import synth


@functools.lru_cache(maxsize=None)
def config(name, **over):
    return synth.make_config(name, **over)


def config_over(name, **over):
    return synth.make_config(name, **over)


@functools.lru_cache(maxsize=None)
def sphere(name, ik=0):
    c = config(name)
    return oracle.sphere(c["rprimd"], c["kpt"][ik], c["ecut"], c["ngfft"])


def rel_err(a, b):
    """max over bands of ||a-b||_2/||b||_2 (SURVEY.md 8(c) reading 17)."""
    a = np.atleast_2d(a); b = np.atleast_2d(b)
    num = np.linalg.norm(a - b, axis=-1); den = np.linalg.norm(b, axis=-1)
    den = np.where(den == 0, 1.0, den)
    return float(np.max(num / den))


def rand_c(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)
