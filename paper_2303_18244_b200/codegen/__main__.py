"""python -m paper_2303_18244_b200.codegen OUTDIR — writes the generated CUDA sources."""
import json
import os
import sys

from . import emit, emit_orbit, emit_orbit5


def main(outdir):
    os.makedirs(outdir, exist_ok=True)
    summary = {}
    for n, name in ((2, "gg_ttx"), (3, "gg_ttxg"), (4, "gg_ttxgg")):
        if n == 4:
            src, info = emit_orbit.emit_orbit_process(name)
        else:
            src, info = emit.emit_single_kernel_process(n, name)
        _write(os.path.join(outdir, "gen_%s.cu" % name), src)
        info.pop("color_num")
        summary[name] = info
    if True:
        files, info = emit_orbit5.emit_orbit5_process("gg_ttxggg")
        for f in os.listdir(outdir):                      # drop files of an earlier generator version
            if f.startswith("gen_gg_ttxggg_") and f not in files:
                os.remove(os.path.join(outdir, f))
        for fn, src in files.items():
            _write(os.path.join(outdir, fn), src)
        info.pop("color_num", None)
        summary["gg_ttxggg"] = info
    _write(os.path.join(outdir, "gen_summary.json"), json.dumps(summary, indent=1) + "\n")
    return summary


def _write(path, text):
    if os.path.exists(path) and open(path).read() == text:
        return                      # keep mtime: no needless recompilation
    with open(path, "w") as f:
        f.write(text)


if __name__ == "__main__":
    print(json.dumps(main(sys.argv[1]), indent=1))
