"""The C-ABI library loads and exports every symbol include/trdmatch.h declares; the header compiles
as plain C and the ctypes mirrors have the C sizes.  No compute calls (runs without a GPU)."""
import ctypes as C
import os
import re
import subprocess
import tempfile

import pytest

from paper_2003_03174_b200 import binding as B, build as Bd

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "trdmatch.h")


@pytest.fixture(scope="module")
def lib():
    Bd.build()
    return B.lib()


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(trd_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert set(names) == set(B.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None
    assert lib.trd_version() == 100


def test_header_is_plain_c_and_struct_sizes_match():
    src = ('#include "trdmatch.h"\n#include <stdio.h>\nint main(void){printf("%zu %zu %zu %zu\\n", sizeof(trd_config),'
           'sizeof(trd_tracks_in), sizeof(trd_tracks_out), sizeof(trd_index_info)); return 0;}\n')
    with tempfile.TemporaryDirectory() as td:
        c = os.path.join(td, "t.c"); exe = os.path.join(td, "t")
        open(c, "w").write(src)
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        sizes = [int(v) for v in subprocess.check_output([exe]).split()]
    assert sizes == [C.sizeof(B.TrdConfig), C.sizeof(B.TrdTracksIn), C.sizeof(B.TrdTracksOut), C.sizeof(B.TrdIndexInfo)]


def test_bad_arguments_are_status_codes_not_crashes(lib, base_cfg):
    h = C.c_void_p()
    assert lib.trd_create(None, C.byref(h)) == B.TRD_E_ARG
    for key, val in (("n_hyp", 0), ("n_hyp", 9), ("n_layers", 7), ("max_snp", 1.5), ("pad_length", 0.0),
                     ("sigma_y", -1.0), ("n_sectors", 0)):
        c = B.make_config(dict(base_cfg, **{key: val}))
        assert lib.trd_create(C.byref(c), C.byref(h)) == B.TRD_E_ARG, key
    c = B.make_config(base_cfg); c.struct_size = 8
    assert lib.trd_create(C.byref(c), C.byref(h)) == B.TRD_E_ARG
    c = B.make_config(dict(base_cfg, layer_x=[300, 313, 313, 338, 351, 364]))
    assert lib.trd_create(C.byref(c), C.byref(h)) == B.TRD_E_ARG
    lib.trd_destroy(None)                                   # NULL is a no-op
    assert lib.trd_match(None, None, None, 0, None) == B.TRD_E_ARG
    assert lib.trd_last_error(None) == b"NULL handle"
    assert lib.trd_device_bytes(None) == 0 and lib.trd_kernel_launches(None) == 0


def test_no_cpu_fallback_without_a_device(lib, base_cfg):
    """Without a CUDA device trd_create must fail loudly (TRD_E_CUDA), never fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(B.TrdError) as e:
        B.trd_create(base_cfg)
    assert e.value.code == B.TRD_E_CUDA


def test_product_path_does_not_reach_the_oracle():
    """Nothing under the package imports or names the oracle."""
    pkg = os.path.join(ROOT, "paper_2003_03174_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dp, f)).read()
                assert "from oracle" not in text and "import oracle" not in text and "trd_oracle" not in text, f


def test_plain_c_program_links_and_calls_the_library(lib):
    """A C99 program (no Python, no torch) links against libtrdmatch.so and uses the ABI: version, argument
    errors, and -- on a machine without a GPU -- the loud TRD_E_CUDA from trd_create."""
    src = r'''
#include "trdmatch.h"
#include <stdio.h>
#include <string.h>
int main(void) {
    trd_config c; trd_handle* h = 0;
    memset(&c, 0, sizeof c);
    if (trd_version() != TRD_VERSION) return 1;
    if (trd_create(0, &h) != TRD_E_ARG) return 2;
    c.struct_size = sizeof c;                       /* all other fields 0: invalid geometry */
    if (trd_create(&c, &h) != TRD_E_ARG || h != 0) return 3;
    c.n_sectors = 18; c.n_stacks = 5; c.n_layers = 6; c.n_hyp = 4;
    { double x[6] = {300, 313, 326, 338, 351, 364}; memcpy(c.layer_x, x, sizeof x); }
    c.z_max = 350; c.pad_length = 8; c.bz_tesla = 0.5; c.sigma_y = 0.04; c.sigma_z = 2.3094; c.sigma_dydx = 0.02;
    c.n_sigma_road = 3; c.n_sigma_angle = 4; c.chi2_cut = 15; c.chi2_penalty = 15; c.max_snp = 0.95;
    { int rc = trd_create(&c, &h); printf("%d\n", rc); if (rc == TRD_OK) { trd_destroy(h); } else if (rc != TRD_E_CUDA) return 4; }
    trd_destroy(0);
    return 0;
}
'''
    with tempfile.TemporaryDirectory() as td:
        cfile = os.path.join(td, "t.c"); exe = os.path.join(td, "t")
        open(cfile, "w").write(src)
        libdir = os.path.dirname(Bd.LIB_PATH)
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), cfile, "-o", exe,
                               "-L", libdir, "-ltrdmatch", "-Wl,-rpath," + libdir])
        out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    import torch
    assert int(out.stdout.split()[0]) == (B.TRD_OK if torch.cuda.is_available() else B.TRD_E_CUDA)
