"""Static check of how ptxas compiled the MMA-issuing warp of a tensor-core kernel (developer utility, not part of libhb):
for every kernel of an object file that holds tcgen05.mma, the code within [first MMA - 1 KB, last MMA + 0.5 KB] is taken
as the issuing region and its R2UR / R2UR.BROADCAST / WARPSYNC / CALL instructions are counted.  Few R2UR per MMA = the
descriptor arithmetic stayed on the uniform datapath (hb_tc_common.cuh, mbar_spin; profiles/r2_issuer_codegen.md).

    python paper_2402_17248_b200/csrc/microbench/issuer_codegen.py paper_2402_17248_b200/build/hb_sur_tc2.o
"""
import sys,re,subprocess,collections
out=subprocess.run(["cuobjdump","-sass",sys.argv[1]],capture_output=True,text=True).stdout
cur=None;fn={}
for line in out.splitlines():
    m=re.search(r"Function : (\S+)",line)
    if m: cur=m.group(1); fn[cur]=[]; continue
    m=re.match(r"\s+/\*([0-9a-f]{4,5})\*/\s+(.*?);",line)
    if cur and m: fn[cur].append((int(m.group(1),16),m.group(2)))
for k,rows in fn.items():
    mma=[a for a,t in rows if "UTCHMMA" in t or "UTCQMMA" in t]
    if not mma: continue
    lo,hi=min(mma)-0x400,max(mma)+0x200
    reg=[re.sub(r"^@!?U?P\d+\s+","",t).split()[0] for a,t in rows if lo<=a<=hi]
    c=collections.Counter(reg)
    name=subprocess.run(["c++filt",k],capture_output=True,text=True).stdout.strip()
    name=re.sub(r"\(.*","",name.replace("(anonymous namespace)::","").replace("void ",""))
    print("%-44s code %6d B  region %5d instr  MMA %3d  R2UR %3d  R2UR.BROADCAST %2d  WARPSYNC %2d  CALL %2d" % (name, rows[-1][0], len(reg), len(mma), c["R2UR"], c["R2UR.BROADCAST"], c["WARPSYNC.ALL"], sum(v for o,v in c.items() if o.startswith("CALL"))))
