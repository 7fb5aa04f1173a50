"""Writes the per-kernel SASS opcode table kept as profiles/sass_opcodes.txt:
    python -m paper_2606_04557_b200.sass_opcodes > profiles/sass_opcodes.txt
(cuobjdump -sass of the built libcas.so; counts the mnemonics that prove the tcgen05 / TMEM / TMA / bulk-reduction
paths -- the list in /opt/skills/guides/B200_PROFILING.md -- per 'Function :' block.)"""
import re
import subprocess
import sys

from . import _build

OPS = ["UTCHMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UBLKCP", "UBLKRED", "UTMAPF", "SYNCS", "MUFU.EX2", "HMMA",
       "USETMAXREG", "ATOMG", "RED"]


def main():
    lib = _build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    demangle = lambda n: subprocess.run(["c++filt", n], capture_output=True, text=True).stdout.strip()
    print("# SASS opcode counts per kernel of libcas.so (sm_100a)\n#\n"
          "# command: python -m paper_2606_04557_b200.sass_opcodes > profiles/sass_opcodes.txt\n"
          "#   (cuobjdump -sass libcas.so, mnemonics counted per 'Function :' block)\n"
          "#   UTCHMMA = tcgen05.mma, LDTM/STTM = tcgen05.ld/st, UTMALDG = TMA tensor load, UBLKCP/UBLKRED = bulk copy /\n"
          "#   bulk reduction (cp.async.bulk / cp.reduce.async.bulk), UTCBAR = tcgen05.commit, SYNCS = mbarrier ops,\n"
          "#   HMMA would be the legacy mma.sync path: none\n#")
    print("%-62s" % "kernel" + "".join("%11s" % o for o in OPS))
    name, counts = None, None

    def flush():
        if name:
            print("%-62s" % name[:62] + "".join("%11d" % counts[o] for o in OPS))

    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            flush()
            name = demangle(m.group(1)).split("(")[0]
            counts = {o: 0 for o in OPS}
            continue
        if counts is None:
            continue
        m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m:
            op = m.group(1)
            for o in OPS:
                if op == o or op.startswith(o + "."):
                    counts[o] += 1
    flush()


if __name__ == "__main__":
    sys.exit(main())
