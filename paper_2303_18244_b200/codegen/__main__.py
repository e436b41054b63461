"""python -m paper_2303_18244_b200.codegen OUTDIR — writes the generated CUDA sources."""
import json
import os
import sys

from . import emit, emit_orbit


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
    if hasattr(emit, "emit_multi_kernel_process"):
        files, info = emit.emit_multi_kernel_process(5, "gg_ttxggg")
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
