"""A plain C program linked against libtpc_tracker.so (tests/c_abi_frame.c): the boundary is usable without Python or
torch.  CPU part: it compiles as C99 against include/tpc_tracker.h and links.  GPU part: it runs cfg1 from a binary
dump and its track / attached-cluster / seed counts equal the oracle's."""
import os
import struct
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _build(tmp_path):
    import paper_2009_07515_b200 as tpc
    lib = tpc.load_library()._name
    exe = str(tmp_path / "c_abi_frame")
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(CUDA, "include"),
           os.path.join(ROOT, "tests", "c_abi_frame.c"), "-o", exe, lib, "-L", os.path.join(CUDA, "lib64"), "-lcudart",
           f"-Wl,-rpath,{os.path.dirname(lib)}", f"-Wl,-rpath,{os.path.join(CUDA, 'lib64')}"]
    subprocess.run(cmd, check=True)
    return exe


def test_c_program_compiles_and_links(tmp_path):
    exe = _build(tmp_path)
    r = subprocess.run([exe], capture_output=True)          # no dump given: usage error, before any CUDA call
    assert r.returncode == 2


@pytest.mark.gpu
def test_c_program_tracks_cfg1_like_the_oracle(tmp_path, cfg1):
    import paper_2009_07515_b200 as tpc
    from oracle import Oracle
    from tpc_synth import default_params
    tf, P = cfg1, default_params(cfg1)
    fkeys = ["tan_half_sector", "bz_tesla", "err_y2", "err_z2", "cell_y", "cell_z", "link_ay", "link_az", "link_b", "link_T",
             "pick_chi2_cut", "max_sinphi", "y_margin", "init_c_ss", "init_c_tt", "init_c_qq"]
    ikeys = ["min_chain_len", "max_gap", "min_tracklet_hits", "min_track_hits"]
    dump = tmp_path / "cfg1.bin"
    with open(dump, "wb") as f:
        f.write(struct.pack("<qii", tf.n, P["n_sectors"], P["n_rows"]))
        f.write(np.asarray(P["row_x"], np.float32).tobytes())
        f.write(np.array([P[k] for k in fkeys], np.float32).tobytes())
        f.write(np.array([P[k] for k in ikeys], np.int32).tobytes())
        f.write(struct.pack("<q", tpc.max_bins_bound(tf.sector, tf.z, P)))
        for a, dt in ((tf.sector, np.uint8), (tf.row, np.uint8), (tf.y, np.float32), (tf.z, np.float32)):
            f.write(np.ascontiguousarray(a, dt).tobytes())
    r = subprocess.run([_build(tmp_path), str(dump)], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    nt, status, attached, seeds = (int(v) for v in r.stdout.split())
    o = Oracle(P).run(tf.sector, tf.row, tf.y, tf.z)
    assert status == 0
    assert nt == o.get("trk_seed").shape[0] > 30
    assert attached == int((o.get("cluster_track") >= 0).sum())
    assert seeds == o.get("seed_head").shape[0]
