"""CPU checks of the boundary: the library loads and exports every symbol include/lsa.h declares,
the ctypes structs match the header's layout, and argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lsa.h")


@pytest.fixture(scope="module")
def lib_path():
    from paper_2606_09079_b200.build import build_library
    return build_library()


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lsa_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_five_path_calls():
    names = _declared()
    for n in ("lsa_init_pools", "lsa_index_select", "lsa_fetch_chunks", "lsa_decode_attention", "lsa_step"):
        assert n in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for n in _declared():
        assert hasattr(lib, n), f"liblsa.so does not export {n}"
    lib.lsa_version.restype = ctypes.c_int
    assert lib.lsa_version() == 4


def test_binding_lists_the_same_symbols(lib_path):
    from paper_2606_09079_b200 import lsa
    assert sorted(lsa.EXPORTS) == _declared()


def test_struct_layout_matches_header(lib_path, tmp_path):
    """Compile include/lsa.h with gcc and compare sizeof/offsetof with the ctypes mirror."""
    import subprocess
    from paper_2606_09079_b200 import lsa
    structs = {"lsa_config": lsa.lsa_config, "lsa_seq_desc": lsa.lsa_seq_desc, "lsa_stats": lsa.lsa_stats, "lsa_l2_config": lsa.lsa_l2_config,
               "lsa_l1_layer": lsa.lsa_l1_layer, "lsa_l1_config": lsa.lsa_l1_config}
    lines = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{HEADER}"', 'int main(void){']
    for name, cls in structs.items():
        lines.append(f'printf("{name} %zu\\n", sizeof({name}));')
        for f, _ in cls._fields_:
            lines.append(f'printf("{name}.{f} %zu\\n", offsetof({name}, {f}));')
    lines.append('return 0;}')
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", str(src), "-o", str(exe)], check=True)
    out = dict(l.split() for l in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines())
    for name, cls in structs.items():
        assert int(out[name]) == ctypes.sizeof(cls), name
        for f, _ in cls._fields_:
            assert int(out[f"{name}.{f}"]) == getattr(cls, f).offset, f"{name}.{f}"


def test_init_rejects_bad_config_without_touching_cuda(lib_path):
    from paper_2606_09079_b200 import lsa
    cfg = lsa.lsa_config()
    cfg.struct_size = 8                         # wrong ABI size
    h = ctypes.c_void_p()
    seq = (lsa.lsa_seq_desc * 1)()
    assert lsa._lib.lsa_init_pools(ctypes.byref(cfg), seq, ctypes.byref(h)) == -1
    assert b"struct_size" in lsa._lib.lsa_last_error(None)
    cfg.struct_size = ctypes.sizeof(lsa.lsa_config)
    cfg.dtype, cfg.B, cfg.H, cfg.D, cfg.C, cfg.W, cfg.Dh, cfg.E, cfg.k, cfg.tau = 1, 1, 64, 512, 128, 16, 64, 64, 0, 64
    assert lsa._lib.lsa_init_pools(ctypes.byref(cfg), seq, ctypes.byref(h)) == -1      # k < 1
    assert b"k must be" in lsa._lib.lsa_last_error(None)
    assert lsa._lib.lsa_step(None, None, None, None, None, None) == -5                  # LSA_ERR_STATE


def test_no_cpu_fallback(lib_path):
    import torch
    from paper_2606_09079_b200 import lsa
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(lsa.LsaError):
        lsa.LsaContext(dtype=0, H=8, D=64, C_=16, W=8, Dh=64, E=64, k=1, tau=4,
                       hot_pool=torch.zeros(4 * 2 * 16 * 64), W_q=torch.zeros(64, 64), seqs=[])
