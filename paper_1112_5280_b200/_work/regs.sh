#!/bin/bash
# prints registers/spills per dslash kernel variant
cd /root/repo/paper_1112_5280_b200
nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -std=c++17 -Xptxas -v -shared -Xcompiler -fPIC -o /tmp/x.so csrc/lqcd.cu 2>&1 | python3 -c "
import sys,re
name=None
for l in sys.stdin:
    m=re.search(r\"Compiling entry function '(\S+)'\",l)
    if m: name=m.group(1)
    m=re.search(r'Used (\d+) registers',l)
    if m and name and 'dslash' in name:
        k=re.search(r'dslash\w*?I([fd])Li(\d+)ELb([01])ELb([01])ELi(\d+)',name)
        print(k.groups() if k else name, 'regs',m.group(1), spill)
    m=re.search(r'(\d+) bytes spill stores',l)
    if m: spill='spill '+m.group(1)
"
