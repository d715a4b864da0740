// Internal: QSS_SCAT(idx, val) of kernel variant 1 -- adds or subtracts `val` to/from one of the 56 register rows
// ct[0..35], cq[0..19] of the Jacobian column, selected by a warp-uniform RUN-TIME index:
//     idx = 2 * row + 1 (subtract) / + 0 (add),  row < 36: ct[row],  row >= 36: cq[row - 36];  idx = 112: nothing.
// The index is resolved by ONE indexed branch (PTX brx.idx -> SASS LDC jump-table entry + BRX) into a DADD on the
// right register, so the column never leaves the register file.  nvcc lowers a C++ switch to a compare tree (the
// NVPTX back end has no jump tables), hence the inline PTX.  Operands %0..%35 = ct[], %36..%55 = cq[], %56 = val,
// %57 = idx.  The text below is written out for QSS_V1_NT = 36, QSS_V1_NQ = 20.
#ifndef QSS_V1_SCATTER_H
#define QSS_V1_SCATTER_H
#define QSS_PM(i) "P" #i ": add.rn.f64 %" #i ", %" #i ", %56; bra.uni LEND;\n\t" \
                  "M" #i ": sub.rn.f64 %" #i ", %" #i ", %56; bra.uni LEND;\n\t"
#define QSS_SCAT(idx, val)                                                                    \
    asm volatile("{\n\t.reg .u32 ix;\n\tmov.u32 ix, %57;\n\t"                                        \
                 "TL: .branchtargets "                                                           \
                 "P0, M0, P1, M1, P2, M2, P3, M3, P4, M4, P5, M5, P6, M6, P7, M7, " \
                 "P8, M8, P9, M9, P10, M10, P11, M11, P12, M12, P13, M13, P14, M14, P15, M15, " \
                 "P16, M16, P17, M17, P18, M18, P19, M19, P20, M20, P21, M21, P22, M22, P23, M23, " \
                 "P24, M24, P25, M25, P26, M26, P27, M27, P28, M28, P29, M29, P30, M30, P31, M31, " \
                 "P32, M32, P33, M33, P34, M34, P35, M35, P36, M36, P37, M37, P38, M38, P39, M39, " \
                 "P40, M40, P41, M41, P42, M42, P43, M43, P44, M44, P45, M45, P46, M46, P47, M47, " \
                 "P48, M48, P49, M49, P50, M50, P51, M51, P52, M52, P53, M53, P54, M54, P55, M55, " \
                 "LEND;\n\t" \
                 "brx.idx.uni ix, TL;\n\t"                                                        \
                 QSS_PM(0) QSS_PM(1) QSS_PM(2) QSS_PM(3) QSS_PM(4) QSS_PM(5) QSS_PM(6) QSS_PM(7) \
                 QSS_PM(8) QSS_PM(9) QSS_PM(10) QSS_PM(11) QSS_PM(12) QSS_PM(13) QSS_PM(14) QSS_PM(15) \
                 QSS_PM(16) QSS_PM(17) QSS_PM(18) QSS_PM(19) QSS_PM(20) QSS_PM(21) QSS_PM(22) QSS_PM(23) \
                 QSS_PM(24) QSS_PM(25) QSS_PM(26) QSS_PM(27) QSS_PM(28) QSS_PM(29) QSS_PM(30) QSS_PM(31) \
                 QSS_PM(32) QSS_PM(33) QSS_PM(34) QSS_PM(35) QSS_PM(36) QSS_PM(37) QSS_PM(38) QSS_PM(39) \
                 QSS_PM(40) QSS_PM(41) QSS_PM(42) QSS_PM(43) QSS_PM(44) QSS_PM(45) QSS_PM(46) QSS_PM(47) \
                 QSS_PM(48) QSS_PM(49) QSS_PM(50) QSS_PM(51) QSS_PM(52) QSS_PM(53) QSS_PM(54) QSS_PM(55) \
                 "LEND:\n\t}"                                                                    \
                 : "+d"(ct[0]), "+d"(ct[1]), "+d"(ct[2]), "+d"(ct[3]), "+d"(ct[4]), "+d"(ct[5]), \
                   "+d"(ct[6]), "+d"(ct[7]), "+d"(ct[8]), "+d"(ct[9]), "+d"(ct[10]), "+d"(ct[11]), \
                   "+d"(ct[12]), "+d"(ct[13]), "+d"(ct[14]), "+d"(ct[15]), "+d"(ct[16]), "+d"(ct[17]), \
                   "+d"(ct[18]), "+d"(ct[19]), "+d"(ct[20]), "+d"(ct[21]), "+d"(ct[22]), "+d"(ct[23]), \
                   "+d"(ct[24]), "+d"(ct[25]), "+d"(ct[26]), "+d"(ct[27]), "+d"(ct[28]), "+d"(ct[29]), \
                   "+d"(ct[30]), "+d"(ct[31]), "+d"(ct[32]), "+d"(ct[33]), "+d"(ct[34]), "+d"(ct[35]), \
                   "+d"(cq[0]), "+d"(cq[1]), "+d"(cq[2]), "+d"(cq[3]), "+d"(cq[4]), "+d"(cq[5]), \
                   "+d"(cq[6]), "+d"(cq[7]), "+d"(cq[8]), "+d"(cq[9]), "+d"(cq[10]), "+d"(cq[11]), \
                   "+d"(cq[12]), "+d"(cq[13]), "+d"(cq[14]), "+d"(cq[15]), "+d"(cq[16]), "+d"(cq[17]), \
                   "+d"(cq[18]), "+d"(cq[19]) \
                 : "d"((double)(val)), "r"((int)(idx)))
#endif
