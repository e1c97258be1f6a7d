"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol include/cf.h declares, the ctypes
mirror of cf_params has the C layout, host-side validation returns the documented status codes (cf_create never
touches the device), and the host Philox of the library is bit-identical to the oracle's.  No compute calls."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cf():
    from paper_2606_01478_b200 import build, cf as m
    build.build()
    m.lib()
    return m


def test_library_exports_every_declared_symbol(cf):
    hdr = open(os.path.join(ROOT, "include", "cf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cf_[a-z_0-9]+)\s*\(", hdr))
    assert {"cf_create", "cf_reset", "cf_step", "cf_get_state"} <= declared
    assert declared == set(cf.EXPORTS), declared ^ set(cf.EXPORTS)
    L = C.CDLL(cf.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name


def test_params_struct_layout_and_defaults_match_the_oracle(cf, cfo):
    for model in (0, 1):
        p = cf.default_params(model)
        assert p.struct_size == C.sizeof(cf.Params)
        o = cfo.make_params(model)
        for name, _ in cf.Params._fields_:
            if name == "struct_size":
                continue
            a, b = getattr(p, name), getattr(o, name)
            a = np.array(a, dtype=np.float64).reshape(-1) if isinstance(a, C.Array) else np.array([a], dtype=np.float64)
            b = np.array(b, dtype=np.float64).reshape(-1) if isinstance(b, C.Array) else np.array([b], dtype=np.float64)
            np.testing.assert_allclose(a, b, rtol=1e-7, err_msg=name)
        assert abs(p.cmd_hi[3] - 0.55) < 1e-7 and abs(p.cmd_lo[2] + np.pi) < 1e-6      # last fields land where C put them
        assert cf.lib().cf_state_dim(model) == (17, 13)[model] and cf.lib().cf_world_param_dim(model) == (14, 11)[model]


def test_workspace_bytes_and_create_validation(cf):
    L = cf.lib()
    p = cf.default_params(0)
    n = L.cf_workspace_bytes(1000, 3, 0, C.byref(p))
    assert n >= 4 * (17 + 14) * 3000 + 4 * 14 * 1000 and n % 256 == 0
    p_obs = cf.default_params(0, dict(n_obstacles=2))
    assert L.cf_workspace_bytes(1000, 3, 0, C.byref(p_obs)) >= n + 4 * 8 * 3000
    h = C.c_void_p()
    fake = C.c_void_p(0x10000000)             # never dereferenced by cf_create

    def create(M, N, model, prm, ws=fake, nbytes=1 << 40):
        return L.cf_create(C.byref(h), M, N, model, C.byref(prm), ws, nbytes)
    assert create(0, 1, 0, p) == cf.E_ARG
    assert create(1 << 20, 1 << 12, 0, p) == cf.E_SHAPE                       # M*N >= 2^31
    assert create(4, 4, 2, p) == cf.E_ARG                                      # bad model
    assert create(4, 4, 0, p, nbytes=16) == cf.E_BUFFER and b"too small" in L.cf_last_error()
    assert create(4, 4, 0, p, ws=C.c_void_p(0x10000010)) == cf.E_BUFFER        # misaligned
    assert create(4, 4, 0, cf.default_params(0, dict(f_att=300.0))) == cf.E_SHAPE
    assert create(4, 4, 1, cf.default_params(1, dict(iface=cf.IF_ROTOR))) == cf.E_UNSUPPORTED
    # values the kernels divide by, or that put NaN into the planes, are refused at create
    lo_bad = [1.0] * 12; lo_bad[6] = 0.0
    assert create(4, 4, 0, cf.default_params(0, dict(rnd_lo=lo_bad))) == cf.E_ARG           # motor time-constant factor 0
    lo_bad = [1.0] * 12; lo_bad[0] = -0.5
    assert create(4, 4, 1, cf.default_params(1, dict(rnd_lo=lo_bad))) == cf.E_ARG           # negative mass factor
    lo_bad = [1.0] * 12; lo_bad[9] = 1.2
    assert create(4, 4, 1, cf.default_params(1, dict(rnd_lo=lo_bad))) == cf.E_ARG           # lo > hi
    assert create(4, 4, 1, cf.default_params(1, dict(cmd_lo=[0.6, -0.5, -3.0, 0.05]))) == cf.E_ARG     # cmd_lo > cmd_hi
    assert create(4, 4, 1, cf.default_params(1, dict(noise_sigma=[0.1, -0.1, 0.0, 0.0]))) == cf.E_ARG
    assert create(4, 4, 0, cf.default_params(0, dict(dist_sigma=-1.0))) == cf.E_ARG
    bad = cf.default_params(0)
    bad.struct_size = 8
    assert create(4, 4, 0, bad) == cf.E_ARG
    assert create(4, 4, 0, p) == cf.OK and h.value
    assert L.cf_step_counter(h) == 0
    # step before reset is refused on the host, before any launch
    assert L.cf_step(h, fake, 1, 1, 1, 0, None, 0) == cf.E_STATE
    name = C.create_string_buffer(128)
    g, b = C.c_int(), C.c_int()
    assert L.cf_set_full(h, None, None, None, None, 1 << 32) == cf.E_SHAPE                    # step counter is 32 bits
    assert L.cf_describe_launch(h, name, 128, C.byref(g), C.byref(b)) == cf.OK
    assert name.value.startswith(b"rollout<FP") and g.value * b.value >= 16
    assert L.cf_destroy(h) == cf.OK


def test_host_philox_bit_exact_with_oracle_and_kat(cf, cfo):
    assert [hex(v) for v in cf.debug_philox(0, [0, 0, 0, 0])] == ["0x6627e8d5", "0xe169c58d", "0xbc57ac4c", "0x9b00dbd8"]
    rng = np.random.default_rng(11)
    for _ in range(300):
        seed = int(rng.integers(0, 2 ** 63)) * 2 + int(rng.integers(0, 2))
        c = [int(v) for v in rng.integers(0, 2 ** 32, 4)]
        assert np.array_equal(cf.debug_philox(seed, c), cfo.philox(seed, c))


def test_product_package_does_not_reach_the_oracle():
    """The product path must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2606_01478_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "cfo.h" not in src and "libcfo" not in src, fn
    for fn in ("cfo.c", "cfo.h", "cfo.py"):
        src = open(os.path.join(ROOT, "oracle", fn)).read()
        assert "paper_2606_01478_b200 import" not in src and "cf_device" not in src and "libcf.so" not in src, fn
