"""The C-ABI library loads, exports every symbol include/tcp.h declares, validates its arguments
and refuses to run without a GPU (no CPU fallback).  CPU only: no compute call is made."""
import ctypes as C
import os
import re

import pytest
import torch

import paper_2401_03041_b200 as tcp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "tcp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tcp_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported_and_bound():
    names = _declared()
    assert len(names) >= 12
    L = tcp.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in tcp.h but not exported by libtcp.so"
        assert hasattr(tcp, n), f"{n} has no Python binding of the same name"
    assert sorted(tcp.EXPORTS) == names


def test_struct_size_matches_library():
    p = tcp.make_params({})
    assert p.struct_size == C.sizeof(tcp.tcp_params)
    assert tcp.tcp_workspace_bytes(8, 8, 8, p) > 0          # the library accepted struct_size
    p.struct_size -= 4
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_workspace_bytes(8, 8, 8, p)
    assert e.value.code == tcp.TCP_EINVAL


def test_workspace_bytes_accounting():
    n = 32
    N = n ** 3
    for thermal, extra in (("lb_d3q7", 14), ("lb_d3q27", 54), ("rk2", 1), ("rk4", 3)):
        for prec, es in (("f64", 8), ("f32", 4)):
            b = tcp.tcp_workspace_bytes(n, n, n, tcp.make_params(dict(thermal=thermal, precision=prec)))
            aa = tcp.tcp_workspace_bytes(n, n, n, tcp.make_params(dict(thermal=thermal, precision=prec, streaming="aa")))
            pops = 54 + (extra // 2 if thermal.startswith("lb") else 0)
            assert abs((b - aa) - pops * N * es) <= 64 * 256      # AA keeps one grid of populations
            fields = 108 + extra + 2 + 2 + 3 + 1            # h, g (x2 grids), thermal, phi x2, T x2, u, q
            planes = 6 * n * n
            assert fields * N * es + planes * es <= b <= fields * N * es + planes * es + 64 * 256


@pytest.mark.parametrize("bad, code", [
    (dict(M=0.0), tcp.TCP_EINVAL), (dict(xi=-1.0), tcp.TCP_EINVAL), (dict(tau_H=-0.5), tcp.TCP_EINVAL),
    (dict(rho_L=0.0), tcp.TCP_EINVAL), (dict(kappa_H=0.0), tcp.TCP_EINVAL),
    (dict(eps_normal=0.0), tcp.TCP_EINVAL), (dict(s_bulk=0.0), tcp.TCP_EINVAL), (dict(s_high=2.0), tcp.TCP_EINVAL),
    (dict(high_rate_equals_shear=2), tcp.TCP_EINVAL),
])
def test_parameter_validation(bad, code):
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_workspace_bytes(8, 8, 8, tcp.make_params(bad))
    assert e.value.code == code
    assert tcp.tcp_last_error()


def test_params_default_matches_the_binding_and_a_zeroed_struct_is_rejected():
    """tcp_params_default (include/tcp.h) fills what the Python binding's PARAM_DEFAULTS documents; a C caller who
    memsets the struct and sets only struct_size gets TCP_EINVAL instead of NaNs (eps_normal = 0, rates 0)."""
    d, b = tcp.tcp_params_default(), tcp.make_params({})
    assert bytes(d) == bytes(b)
    z = tcp.tcp_params()
    z.struct_size = C.sizeof(tcp.tcp_params)
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_workspace_bytes(8, 8, 8, z)
    assert e.value.code == tcp.TCP_EINVAL


def test_extent_validation():
    p = tcp.make_params(dict(bc=("periodic", "walls", "periodic")))
    for dims in ((0, 4, 4), (4, 1, 4), (2048, 2048, 2048), (800, 800, 800)):   # 800^3: 10 N >= 2^32
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_workspace_bytes(*dims, p)
        assert e.value.code == tcp.TCP_EINVAL
    assert tcp.tcp_workspace_bytes(1, 2, 1, p) > 0
    # any s_high is accepted (general central-moment mode), also together with BGK mode (where it is ignored)
    assert tcp.tcp_workspace_bytes(4, 4, 4, tcp.make_params(dict(s_high=1.3))) > 0
    assert tcp.tcp_workspace_bytes(4, 4, 4, tcp.make_params(dict(s_high=1.3, high_rate_equals_shear=1))) > 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback():
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_create(8, 8, 8, tcp.make_params({}))
    assert e.value.code == tcp.TCP_ECUDA
    with pytest.raises(RuntimeError):
        tcp.Simulation(8, 8, 8, {})


def test_product_does_not_import_oracle():
    """The product path shares nothing with oracle/: no import, include or symbol of it."""
    pkg = os.path.join(ROOT, "paper_2401_03041_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+\.*oracle", txt, flags=re.M), f
                assert not re.search(r"#include\s+[\"<].*oracle", txt), f
                assert "tcpo" not in txt, f
