"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds for sm_100a, loads and
exports every symbol include/spegg.h declares; parameter validation and workspace sizing work
without a GPU (no compute calls)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1603_09255_b200 import binding as b
    from paper_1603_09255_b200 import build
    build.build()
    b.load()
    return b


def test_library_exports_every_declared_symbol(binding):
    hdr = open(os.path.join(ROOT, "include", "spegg.h")).read()
    declared = set(re.findall(r"\b(spegg_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    lib = binding.load()
    for name in declared:
        assert hasattr(lib, name), name


def test_every_entry_point_cites_its_passage():
    """each call declared in include/spegg.h cites the passage of the paper that defines
    the operation -- the comment block directly above the declaration names a PAPER.md line."""
    hdr = open(os.path.join(ROOT, "include", "spegg.h")).read()
    decls = list(re.finditer(r"^(?:int|void|const char \*)\s*(spegg_[a-z_]+)\(", hdr, re.M))
    assert len(decls) >= 14
    for m in decls:
        before = hdr[:m.start()].rstrip()
        assert before.endswith("*/"), m.group(1)
        comment = before[before.rindex("/*"):]
        assert re.search(r"PAPER\.md:\d+", comment), "%s: no passage cited" % m.group(1)


def test_struct_sizes_match_header(binding):
    import ctypes as C
    # spegg_create checks struct_size; mirror the arithmetic of the C layout here
    assert C.sizeof(binding.LogEntry) == 64
    assert C.sizeof(binding.Params) == 48
    assert C.sizeof(binding.SpeciesParams) == 240   # + resid_sd, adult_survival (version 2), mate_skew (3), encounters (4), separate_sexes (5), fec_cost (6), assort (7), mother_skew (8), monogamy (9)


def test_workspace_bytes_and_validation(binding):
    from paper_1603_09255_b200 import workloads
    c3 = workloads.config(3)
    n = binding.workspace_bytes(c3)
    cap, row = c3["species"][0]["capacity"], 256
    assert n >= 3 * cap * row and n < 4 * cap * row  # two population buffers + staging + indices
    assert binding.workspace_bytes(workloads.config(5)) < 8 * 2 ** 30
    for mutate in (lambda c: c["species"][0].update(mu=2.0),
                   lambda c: c["species"][0].update(capacity=0),
                   lambda c: c["species"][0].update(chrom_len=[512, 256], xover_mean=[1.0, 1.0]),
                   lambda c: c["species"][0].update(K=0.0),
                   lambda c: c["species"][0].update(mate_skew=float("nan")),
                   lambda c: c["species"][0].update(predation=dict(attack=0.1, predator=0, encounters=2)),   # no such consumer
                   lambda c: c["species"][0].update(adult_survival=1.5)):
        c = workloads.config(3, scale=0.01)
        mutate(c)
        with pytest.raises(binding.SpeggError) as e:
            binding.workspace_bytes(c)
        assert e.value.code == binding.EINVAL
    assert binding.load().spegg_strerror(binding.EINVAL) == b"invalid parameter"


def test_no_library_dependencies_on_thrust_cub_or_oracle():
    # north_star: hand-written kernels, no Thrust/CUB; the product path never touches oracle/
    src_dir = os.path.join(ROOT, "paper_1603_09255_b200")
    for dirpath, _, files in os.walk(src_dir):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h", ".py")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"#include\s*<(thrust|cub)/", txt), f
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, re.M), f
                assert "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1603_09255_b200", txt, re.M), f
            assert not re.search(r"#include\s*\"[^\"]*spegg_(device|internal|kernels|fused)", txt), f


def test_bench_workloads_and_variants_validate(binding):
    """bench.py's workloads (every configuration, every --variant, the sweep sizes of the NEXT-4 series
    and --k-scale) are accepted by the library's validation (host logic only: spegg_workspace_bytes)."""
    import bench
    try:
        for which in (1, 2, 3, 4, 5, 6):
            for variant in sorted(bench.VARIANTS):
                if variant == "encounters" and which != 4:
                    continue
                cfg = bench.workload(which, variant=variant)
                assert binding.workspace_bytes(cfg) > 0, (which, variant)
        for patches, per in ((1, 50_000), (100, 50_000), (10_000, 1_000)):
            bench.SWEEP.update(patches=patches, per_patch=per)
            cfg = bench.workload(6, variant="overlap")
            assert cfg["grid"] == (patches, 1) and cfg["n0"][0] == patches * per
            assert binding.workspace_bytes(cfg) > 0
        bench.SWEEP.update(patches=16, per_patch=50_000, k_scale=0.5)
        cfg = bench.workload(3)
        assert cfg["species"][0]["K"] == 500_000.0 and "K x 0.5" in cfg["name"]
    finally:
        bench.SWEEP.update(patches=16, per_patch=50_000, k_scale=1.0)
