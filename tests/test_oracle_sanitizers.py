"""the CPU oracle once under AddressSanitizer + UndefinedBehaviorSanitizer (no GPU).

The oracle is compiled to a separate shared object with -fsanitize=address,undefined -fno-sanitize-recover and driven, in
a child interpreter with the ASan runtime preloaded, through config 1 in both candidate modes (brute force on a pixel
sample, tile-culled on the full frame) forward + backward, a sky + normal-map render, the feature pass, the T1 reference
list and the per-ray segment list.  Any heap overflow, use after free, misaligned access, signed overflow or out-of-range
shift aborts the child with a non-zero exit code."""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = textwrap.dedent("""
    import sys
    sys.path.insert(0, %(root)r)
    import numpy as np
    import dvx_scenes as S
    from oracle import oracle as O
    O._LIB = %(lib)r                      # the sanitized build, never the timed one
    O.build = lambda force=False: O._LIB
    s = S.make_config(1)
    cam = s.cameras[0]
    g = s.image_grads(0, 1e-2, 1e-3, 1e-2)
    mask = np.zeros((cam.height, cam.width), dtype=np.uint8)
    mask[::7, ::5] = 1
    a = O.render(s, mode=0, mask=mask, grads_in=g)
    b = O.render(s, mode=1, grads_in=g)
    m = mask.astype(bool)
    assert np.array_equal(a["rgb"][m], b["rgb"][m])
    tex = np.random.RandomState(0).uniform(size=(6, 12, 3))
    g["normal"] = np.random.RandomState(1).normal(size=(cam.height, cam.width, 3))
    c = O.render(s, mode=1, mask=mask, grads_in=g, sky=tex)
    feats = [np.random.RandomState(2 + n).uniform(size=(t.n_voxels, 5)) for n, t in enumerate(s.octrees)]
    img = np.random.RandomState(9).uniform(size=(cam.height, cam.width, 5))
    O.render_features(s, feats=feats, img=img, mode=1, mask=mask)
    assert len(O.tile_hit_list(s, 3, 3, 0, 0)) >= 0
    O.ray_segments(s, 64, 60)
    small = S.tiny_random_scene(3)
    O.render(small, grads_in=small.image_grads(0, 1.0, 0.3, 1.0), t_stop=1e-4)
    print("sanitized oracle ok", float(b["alpha"].max()))
""")


@pytest.mark.slow
def test_oracle_under_asan_ubsan(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("gcc has no libasan here")
    lib = str(tmp_path / "libdvx_oracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-fopenmp", "-std=c99", "-shared", "-fPIC", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-o", lib,
                           os.path.join(ROOT, "oracle", "dvx_oracle.c"), "-lm"])
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4")
    r = subprocess.run([sys.executable, "-c", CHILD % {"root": ROOT, "lib": lib}], capture_output=True, text=True, env=env,
                       timeout=900)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert "sanitized oracle ok" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
