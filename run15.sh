#!/bin/bash
cd /root/repo/_work
echo "## h3"; ./kb_h3 2 16384 1 4096 5 1e14; ./kb_h3 3 1024 1024 256 3 1e11
for v in i1 i2 i3; do echo "## $v"; ./kb_$v 3 1024 1024 256 3 1e11; done
