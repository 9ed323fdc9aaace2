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


C_PROGRAM = r'''
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
    { int rc = trd_create(&c, &h); printf("%d\n", rc); if (rc == TRD_E_CUDA) { trd_destroy(0); return 0; } if (rc != TRD_OK) return 4; }
    {   /* two infinite-momentum tracks (q/pT = 0) along x: track 0 in sector 4 at y = 1, z = 4; track 1 in sector 9 at
           y = -2, z = -12 with no tracklet in layer 3.  Tracklets sit exactly on the lines, z on pad-row centres. */
        float ty[12], tz[12], td[12]; int32_t tc[12]; int n = 0, l, k;
        float par[5][2] = {{1.0f, -2.0f}, {4.0f, -12.0f}, {0.0f, 0.0f}, {0.0f, 0.0f}, {0.0f, 0.0f}};
        float cov[15][2]; float x[2] = {247.0f, 247.0f}; int32_t sec[2] = {4, 9};
        float opar[5][2], ocov[15][2], ox[2], ochi2[2]; int32_t oidx[TRD_MAX_LAYERS][2], osec[2], onm[2], oev[2];
        trd_tracks_in in; trd_tracks_out out;
        for (l = 0; l < 6; ++l) { ty[n] = 1.0f; tz[n] = 4.0f; td[n] = 0.0f; tc[n] = 4 * 30 + 2 * 6 + l; ++n; }
        for (l = 0; l < 6; ++l) { if (l == 3) continue; ty[n] = -2.0f; tz[n] = -12.0f; td[n] = 0.0f; tc[n] = 9 * 30 + 2 * 6 + l; ++n; }
        ty[n] = 1.0f; tz[n] = 4.0f; td[n] = 0.0f; tc[n] = 5 * 30 + 2 * 6 + 2; ++n;       /* same place, other sector: never a candidate */
        memset(cov, 0, sizeof cov);
        for (k = 0; k < 2; ++k) { cov[0][k] = 0.01f; cov[2][k] = 0.01f; cov[5][k] = 1e-6f; cov[9][k] = 1e-6f; cov[14][k] = 1e-4f; }
        memset(&in, 0, sizeof in); memset(&out, 0, sizeof out);
        for (k = 0; k < 5; ++k) { in.par[k] = par[k]; out.par[k] = opar[k]; }
        for (k = 0; k < 15; ++k) { in.cov[k] = cov[k]; out.cov[k] = ocov[k]; }
        in.x = x; in.sector = sec;
        for (l = 0; l < TRD_MAX_LAYERS; ++l) out.tracklet_idx[l] = oidx[l];
        out.x = ox; out.sector = osec; out.chi2 = ochi2; out.n_matched = onm; out.n_cand_evals = oev;
        if (trd_load_tracklets_host(h, ty, tz, td, tc, n, 0) != TRD_OK) { printf("%s\n", trd_last_error(h)); return 5; }
        if (trd_match_host(h, &in, &out, 2, 0) != TRD_OK) { printf("%s\n", trd_last_error(h)); return 6; }
        for (l = 0; l < 6; ++l) if (oidx[l][0] != l) return 7;
        for (l = 0; l < 6; ++l) if (oidx[l][1] != (l == 3 ? -1 : (l < 3 ? 6 + l : 5 + l))) return 8;
        if (onm[0] != 6 || onm[1] != 5 || osec[0] != 4 || osec[1] != 9 || ox[0] != 364.0f) return 9;
        if (!(ochi2[0] >= 0.0f && ochi2[0] < 1e-6f) || opar[0][0] != 1.0f || opar[1][1] != -12.0f) return 10;
        if (oev[0] < 6 || oev[1] < 5 || trd_kernel_launches(h) < 2) return 11;      /* every hypothesis counts its own */
    }
    trd_destroy(h);
    trd_destroy(0);
    return 0;
}
'''


def _run_c_program():
    with tempfile.TemporaryDirectory() as td:
        cfile = os.path.join(td, "t.c"); exe = os.path.join(td, "t")
        open(cfile, "w").write(C_PROGRAM)
        libdir = os.path.dirname(Bd.LIB_PATH)
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), cfile, "-o", exe,
                               "-L", libdir, "-ltrdmatch", "-Wl,-rpath," + libdir])
        return subprocess.run([exe], capture_output=True, text=True)


def test_plain_c_program_links_and_calls_the_library(lib):
    """A C99 program (no Python, no torch) links against libtrdmatch.so and uses the ABI: version, argument
    errors, and -- on a machine without a GPU -- the loud TRD_E_CUDA from trd_create.  With a GPU it runs the whole
    path through C: trd_load_tracklets_host + trd_match_host on two straight tracks and twelve tracklets placed on
    their lines (one of them in a neighbouring sector, one layer left out), and checks the chains that come back."""
    out = _run_c_program()
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    import torch
    assert int(out.stdout.split()[0]) == (B.TRD_OK if torch.cuda.is_available() else B.TRD_E_CUDA)


@pytest.mark.gpu
def test_plain_c_program_runs_load_and_match_on_the_gpu(lib):
    """The same C program on the GPU box: trd_create succeeds, so it goes on to trd_load_tracklets_host and
    trd_match_host and checks the chains itself (exit code 0 only if they are right)."""
    out = _run_c_program()
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    assert int(out.stdout.split()[0]) == B.TRD_OK
