"""CPU-side checks of the C ABI: the shared library loads, exports every symbol that
include/ddhf.h declares, and the ctypes mirror of its structs has the C layout."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "include", "ddhf.h")


@pytest.fixture(scope="module")
def built_lib():
    from paper_2603_08386_b200 import build
    return build.build()


def _declared_functions():
    text = open(HDR).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ddhf_[a-z_0-9]+)\s*\(", text)))


def test_header_functions_are_exported(built_lib):
    from paper_2603_08386_b200 import binding
    names = _declared_functions()
    assert len(names) >= 8
    assert sorted(binding.EXPORTS) == names
    lib = C.CDLL(built_lib)
    for n in names:
        assert hasattr(lib, n), f"{n} not exported"
    out = subprocess.check_output(["nm", "-D", "--defined-only", built_lib], text=True)
    exported = set(re.findall(r" T (ddhf_\w+)", out))
    assert exported == set(names), exported ^ set(names)


def test_struct_layout_matches_c(tmp_path):
    from paper_2603_08386_b200 import binding, workloads
    src = tmp_path / "layout.c"
    src.write_text(r'''
#include <stdio.h>
#include <stddef.h>
#include "ddhf.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu\n", sizeof(ddhf_event), sizeof(ddhf_box), sizeof(ddhf_config),
         sizeof(ddhf_outputs), sizeof(ddhf_host_outputs));
  printf("%zu %zu %zu %zu %zu %zu\n", offsetof(ddhf_config, f_min_hz), offsetof(ddhf_config, n_f0),
         offsetof(ddhf_config, tau_sf), offsetof(ddhf_config, max_events),
         offsetof(ddhf_config, flags), offsetof(ddhf_event, t_us));
  return 0; }''')
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           str(src), "-o", str(exe)])
    l1, l2 = subprocess.check_output([str(exe)], text=True).split("\n")[:2]
    sizes = [int(x) for x in l1.split()]
    offs = [int(x) for x in l2.split()]
    assert sizes == [workloads.EVENT_DTYPE.itemsize, binding.BOX_DTYPE.itemsize,
                     C.sizeof(binding.DdhfConfig), C.sizeof(binding.DdhfOutputs),
                     C.sizeof(binding.DdhfHostOutputs)]
    cfg = binding.DdhfConfig
    assert offs == [cfg.f_min_hz.offset, cfg.n_f0.offset, cfg.tau_sf.offset, cfg.max_events.offset,
                    cfg.flags.offset, workloads.EVENT_DTYPE.fields["t"][1]]


def test_header_compiles_as_c_and_cpp(tmp_path):
    for comp, ext in (("gcc", "c"), ("g++", "cpp")):
        f = tmp_path / f"t.{ext}"
        f.write_text('#include "ddhf.h"\nint main(void) { return DDHF_N_COUNTERS == 16 ? 0 : 1; }\n')
        subprocess.check_call([comp, "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(f),
                               "-o", str(tmp_path / f"t_{ext}")])


def test_version_and_no_device_error(built_lib):
    """ddhf_version works without a GPU; ddhf_create fails loudly (no CPU fallback)."""
    import torch
    from paper_2603_08386_b200 import binding, workloads
    assert "sm_100a" in binding.ddhf_version()
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    cfg = binding.make_config(workloads.preset(1), max_events=100)
    with pytest.raises(binding.DdhfError) as e:
        binding.ddhf_create(cfg)
    assert e.value.code == binding.DDHF_E_CUDA
    with pytest.raises(RuntimeError):
        binding.Detector(workloads.preset(1), max_events=100)


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or anything under _work/)."""
    pkg = os.path.join(ROOT, "paper_2603_08386_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "ddhf_oracle" not in text and "_work/" not in text, f
