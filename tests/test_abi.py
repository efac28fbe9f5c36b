"""The C-ABI library loads and exports every symbol include/rt_tddft.h declares; without a GPU it fails loudly
(no CPU fallback).  No compute calls here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2410_09189_b200.build import build
    return build()


def test_header_symbols_exported(built):
    hdr = open(os.path.join(ROOT, "include", "rt_tddft.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", hdr))
    assert {"rt_create", "rt_set_field", "rt_step", "rt_get_dipole", "rt_get_density"} <= declared
    lib = ctypes.CDLL(built)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in rt_tddft.h but not exported"
    from paper_2410_09189_b200 import binding
    assert set(binding.SYMBOLS) == declared


def test_config_struct_layout(built):
    from paper_2410_09189_b200 import binding
    # values printed by a C program (sizeof / offsetof on include/rt_tddft.h, x86-64 SysV ABI)
    assert ctypes.sizeof(binding.rt_config) == 176 and ctypes.sizeof(binding.rt_slab_buffers) == 48
    assert ctypes.sizeof(binding.rt_shard_buffers) == 64 and binding.rt_shard_buffers.block_count.offset == 40
    assert binding.rt_config.dt.offset == 32 and binding.rt_config.E0.offset == 72
    assert binding.rt_config.flags.offset == 96 and binding.rt_config.stream.offset == 104
    assert binding.rt_config.propagator.offset == 112 and binding.rt_config.max_order.offset == 116
    assert binding.rt_config.dP_thrs.offset == 120 and binding.rt_config.H_thrs.offset == 128
    assert binding.rt_config.max_hupdates.offset == 136
    assert binding.rt_config.slab_x0.offset == 140 and binding.rt_config.slab_nx.offset == 144
    assert binding.rt_config.history.offset == 148
    assert binding.rt_config.prop_shards.offset == 152 and binding.rt_config.prop_shard.offset == 156
    assert binding.rt_config.magnus_order.offset == 160 and binding.rt_config.xc_functional.offset == 164
    assert binding.rt_config.fd_order.offset == 168


def test_no_cpu_fallback(built):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2410_09189_b200 import binding
    phi = np.zeros((2, 8))
    with pytest.raises(binding.RTError) as ei:
        binding.RTTDDFT((2, 2, 2), 0.5, phi, np.zeros(2), np.zeros(2), 0.1, stream=0)
    assert ei.value.code == binding.RT_ECUDA


def test_bad_arguments_rejected(built):
    from paper_2410_09189_b200 import binding
    phi = np.zeros((2, 8))
    with pytest.raises(binding.RTError) as ei:
        binding.RTTDDFT((2, 2, 2), 0.5, phi, np.zeros(2), np.array([3.0, 0.0]), 0.1, stream=0)
    assert ei.value.code == binding.RT_EINVAL
    with pytest.raises(binding.RTError) as ei:
        binding.RTTDDFT((1, 2, 2), 0.5, phi, np.zeros(2), np.zeros(2), 0.1, stream=0)
    assert ei.value.code == binding.RT_EINVAL
